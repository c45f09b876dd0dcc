// Fused decode + render kernel, warp-per-tile variant (sm_100a) -- the default of hmlfc_render.
//
// PAPER.md:289-293 (decoding procedure): "collect the required BISE compressed SRV blocks from the
// top level to the bottom level.  Using the block indices, we infer whether a block belongs to the
// predictive SRV images ... The motion vector values for the corresponding block are decoded" and
// "As a block of pixels are decoded, our method benefits any LF rendering scheme by
// providing fast access to neighboring pixels for interpolation".
//
// ONE WARP renders a 16 x 8 tile of one output view (4 consecutive pixels per lane) out of a
// private shared-memory workspace; warps never wait for each other (no CTA barrier after the
// digit-table load), so the SM hides the latency of one warp's narrow phases behind the others.
// The tree walk is organised the way the paper states it -- per BLOCK -- and compacted so that the
// expensive steps run on full warps over non-empty blocks only (at ~40 dB most blocks are empty):
//   A   ray set-up (screen coordinates once per column / row, shared by shuffles); bounding box of
//       the tile's 16-tap footprints in (u,v,s,t);
//   S   the box's SRV planes: per level L the rectangle of planes (u>>L, v>>L) -- level >= 1 planes
//       are shared by the 2^L x 2^L views below them, so each is visited once per tile;
//   B1  one lane per (plane, channel, block) item: ONE 128-bit flag/rank record load, test the
//       res / pred bits; non-empty items are compacted (ballot) into a record list;
//   B2  one lane per record: decode the block's motion record once (BISE), clip the block against
//       the footprint box, emit one task per needed value (warp scan);
//   R   one lane per (view, sample) cell of the box: the top-level RKV sample initialises the cell's
//       (Y, Co, Cg) accumulator in shared memory;
//   B3  one lane per value task: BISE decode_at of the stored value, motion re-compensation from
//       the reference SRV (flag/rank + BISE decode_at), added (shared-memory atomics) to the cell of
//       every view of the box that lies below the plane;
//   B4  one lane per cell, in place: inverse YCoCg-R, clamp -> float RGB;
//   C   every pixel gathers its 16 taps from the patch (128-bit loads), blends with packed fp32 FMAs,
//       and the lane's 4 pixels leave as three 32-bit stores.
// A tile whose footprint exceeds the workspace is split by lane ranges (rows 8 -> 4 -> 2 -> 1, half rows, single
// lanes); a single lane that still does not fit (strong minification) is rendered by 16 direct sample decodes per pixel.  All
// paths produce identical bytes.
#include "hmlfc_kernels.cuh"

namespace hmlfc {

namespace {

constexpr int kTileH = 8;        // tile height: lane = row * 4 + column group, kPPL consecutive pixels per lane
constexpr int kMaxSlots = 40;    // SRV planes of one footprint, all levels
constexpr int kMaxViews = 16;    // views of one footprint
constexpr int kMaxItems = 8192;

// Compile-time shape of one instantiation: tile = (4 PPL) x 8 output pixels per warp, and the capacities of the
// warp's shared-memory workspace.
template <int PPL_, int WARPS_, int REC_, int TASK_, int CELL_, int MINB_>
struct Cfg {
    static constexpr int kPPL = PPL_, kTileW = 4 * PPL_;
    static constexpr int kWarps = WARPS_;   // warps (= tiles) per CTA
    static constexpr int kRecCap = REC_;    // non-empty (plane, channel, block) records per chunk
    static constexpr int kTaskCap = TASK_;  // value tasks per chunk
    static constexpr int kCellCap = CELL_;  // (view, sample) cells: int4 accumulators, then float4 RGB in place
    static constexpr int kMinBlocks = MINB_;
};

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

__device__ const DigitLut g_warp_digit_lut = make_digit_lut();

// n / d for n * d < 2^32 by one multiply-high (m == 0 encodes d == 1)
__device__ __forceinline__ uint32_t magic_of(uint32_t d) { return d <= 1u ? 0u : 0xFFFFFFFFu / d + 1u; }
__device__ __forceinline__ uint32_t fdiv(uint32_t n, uint32_t m) { return m ? __umulhi(n, m) : n; }

// bits [pos, pos+n) of an LSB-first 32-bit word string, n <= 16
__device__ __forceinline__ uint32_t bits_at(const uint32_t *__restrict__ w, uint32_t pos, uint32_t n)
{
    const uint32_t *p = w + (pos >> 5);
    return __funnelshift_r(__ldg(p), __ldg(p + 1), pos & 31u) & ((1u << n) - 1u);
}

// BISE decode_at (layout in DESIGN.md section 4) with the digit tables in shared memory
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

// The same decode without control flow (plain = groups of one value with an empty digit word): every lane of a
// warp issues the same loads, so independent decodes overlap and lanes with different layouts do not serialise.
__device__ __forceinline__ uint32_t bise_at_uniform(const uint32_t *__restrict__ w, uint32_t i, uint32_t layout, uint32_t m,
                                                    const uint16_t *__restrict__ lut)
{
    const bool plain = layout == 0u, trit = layout == 1u;
    const uint32_t G = plain ? 1u : (trit ? 5u : 3u), hb = plain ? 0u : (trit ? 8u : 7u);
    const uint32_t g = plain ? i : (trit ? (__umulhi(i, 0xCCCCCCCDu) >> 2) : (__umulhi(i, 0xAAAAAAABu) >> 1));
    const uint32_t k = i - G * g;
    const uint32_t gb = g * (hb + G * m);
    const uint32_t head = bits_at(w, gb, hb);  // plain: 0 bits -> 0, and the quint table maps 0 to digit 0
    const uint32_t low = bits_at(w, gb + hb + k * m, m);
    const uint32_t dig = ((uint32_t)lut[(trit ? 0u : 256u) + head] >> (k * (trit ? 2u : 3u))) & (trit ? 3u : 7u);
    return (dig << m) | low;
}

template <class C>
struct Queues {
    uint4 rec[C::kRecCap][2];
    uint16_t task[C::kTaskCap];
};

template <class C>
struct WarpWs {
    union {
        int4 acc[C::kCellCap];      // {Y, Co, Cg, -} per (view, sample) while the levels are summed
        float4 rgb[C::kCellCap];    // {R, G, B, 0} afterwards
    } cell;
    Queues<C> q;
    uint4 slotinfo[kMaxSlots];      // {pc index of channel 0, pc index of the reference plane's channel 0, predictive, views below}
    int lvl_base[kMaxLevels], lvl_pu0[kMaxLevels], lvl_pv0[kMaxLevels], lvl_nu[kMaxLevels];
};

struct PixTaps {  // one output pixel's 16-tap footprint
    uint32_t uv;  // u0 | v0 << 12 | du << 24 | dv << 25   (0xFFFFFFFF: the ray misses the slab)
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

// quadrilinear blend of 16 float RGB taps fetched by idx(a, b): a = view (bit0 u, bit1 v), b = pixel (bit0 s, bit1 t)
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

// strong minification: the footprint of even one tile row exceeds the workspace -> 16 direct sample decodes
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

template <class C>
__global__ void __launch_bounds__(C::kWarps * 32, C::kMinBlocks)
render_warp_kernel(const __grid_constant__ DevStream S, const Camera *__restrict__ cams, int W, int H, uint8_t *__restrict__ out, int out_aligned,
                   int tiles_x, int tiles_per_view)
{
    constexpr int kPPL = C::kPPL, kTileW = C::kTileW, kWarps = C::kWarps;
    constexpr int kRecCap = C::kRecCap, kTaskCap = C::kTaskCap, kCellCap = C::kCellCap;
    static_assert(kRecCap >= 32 && (kRecCap << 6) <= 65536 && kTaskCap >= 64, "queue capacities");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint16_t lut[384];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int q = threadIdx.x; q < 192; q += kWarps * 32)
        reinterpret_cast<uint32_t *>(lut)[q] = reinterpret_cast<const uint32_t *>(g_warp_digit_lut.v)[q];
    __syncthreads();  // the only CTA-wide barrier

    const int tile = blockIdx.x * kWarps + warp;
    if (tile >= tiles_per_view) return;
    WarpWs<C> &ws = reinterpret_cast<WarpWs<C> *>(smem_raw)[warp];
    const int view = blockIdx.y;
    const int ty = tile / tiles_x, tx = tile - ty * tiles_x;
    const int ry = lane >> 2, cg = lane & 3;
    const int x0 = tx * kTileW + cg * kPPL, y = ty * kTileH + ry;
    const uint32_t FULL = 0xffffffffu;
    const int h = S.h, logB = S.logB, Bm1 = S.B - 1;

    // ---------------------------------------------------------------- A: rays of the lane's 4 pixels
    PixTaps pt[kPPL];
    {
        const Camera cam = cams[view];
        const float pxl = ray_screen(cam.tan_half_x, W, tx * kTileW + (lane & (kTileW - 1)));
        const float pyl = ray_screen(cam.tan_half_y, H, ty * kTileH + (lane & 7));
        const float py = __shfl_sync(FULL, pyl, ry);
#pragma unroll
        for (int p = 0; p < kPPL; ++p) {
            const float px = __shfl_sync(FULL, pxl, cg * kPPL + p);
            pt[p].uv = 0xFFFFFFFFu; pt[p].st = 0u;
            pt[p].fu = pt[p].fv = pt[p].fs = pt[p].ft = 0.f;
            if (x0 + p < W && y < H) {
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
    const uint32_t bg = (uint32_t)S.bg[0] | ((uint32_t)S.bg[1] << 8) | ((uint32_t)S.bg[2] << 16);
    uint32_t rgb[kPPL];
#pragma unroll
    for (int p = 0; p < kPPL; ++p) rgb[p] = bg;

    // ---------------------------------------------------------------- row ranges: whole tile first, halved while the footprint does not fit
    // lane ranges: the whole tile (32 lanes) first; a range whose footprint does not fit the workspace is halved
    // (rows 0-3 | 4-7, row pairs, rows, half rows, single lanes) and the halves are processed one after the other
    int row0 = 0, span = 32;
    while (row0 < 32) {
        const bool inr = lane >= row0 && lane < row0 + span;
        int lo[4] = {0x7fffffff, 0x7fffffff, 0x7fffffff, 0x7fffffff}, hi[4] = {-1, -1, -1, -1};
        if (inr) {
#pragma unroll
            for (int p = 0; p < kPPL; ++p)
                if (pt[p].uv != 0xFFFFFFFFu) {
                    const int u0 = pt[p].uv & 0xFFF, v0 = (pt[p].uv >> 12) & 0xFFF, s0 = pt[p].st & 0x3FFF, t0 = (pt[p].st >> 14) & 0x3FFF;
                    lo[0] = min(lo[0], u0); hi[0] = max(hi[0], u0 + (int)((pt[p].uv >> 24) & 1u));
                    lo[1] = min(lo[1], v0); hi[1] = max(hi[1], v0 + (int)((pt[p].uv >> 25) & 1u));
                    lo[2] = min(lo[2], s0); hi[2] = max(hi[2], s0 + (int)((pt[p].st >> 28) & 1u));
                    lo[3] = min(lo[3], t0); hi[3] = max(hi[3], t0 + (int)((pt[p].st >> 29) & 1u));
                }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            lo[q] = __reduce_min_sync(FULL, lo[q]);
            hi[q] = __reduce_max_sync(FULL, hi[q]);
        }
        bool done = hi[0] < 0;  // no ray of the range hits the slab: background only
        if (!done) {
            const int bu0 = lo[0], bv0 = lo[1], bs0 = lo[2], bt0 = lo[3];
            const int nu = hi[0] - lo[0] + 1, nv = hi[1] - lo[1] + 1, ns = hi[2] - lo[2] + 1, nt = hi[3] - lo[3] + 1;
            const int bx0 = lo[2] >> logB, by0 = lo[3] >> logB;
            const int nbw = (hi[2] >> logB) - bx0 + 1, nbh = (hi[3] >> logB) - by0 + 1;
            // S (part 1): per level the rectangle of planes; lane L owns level L
            int pu0 = 0, pv0 = 0, nuL = 0, cntL = 0;
            if (lane < h) {
                pu0 = lo[0] >> lane; pv0 = lo[1] >> lane;
                nuL = (hi[0] >> lane) - pu0 + 1;
                cntL = nuL * ((hi[1] >> lane) - pv0 + 1);
            }
            int incl = cntL;
#pragma unroll
            for (int o = 1; o < kMaxLevels; o <<= 1) {
                const int n = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += n;
            }
            const int nslots = __shfl_sync(FULL, incl, h - 1);
            const long long nsamp_l = (long long)ns * nt, nviews_l = (long long)nu * nv, nblk_l = (long long)nbw * nbh;
            const bool fits = nu <= 8 && nv <= 8 && nviews_l <= kMaxViews && nslots <= kMaxSlots && nbw <= 32 && nbh <= 32 &&
                              nviews_l * nsamp_l <= kCellCap && nslots * 3 * nblk_l <= kMaxItems;
            if (fits) {
                const int nsamp = (int)nsamp_l, nviews = (int)nviews_l, nblkbox = (int)nblk_l, nitems = nslots * 3 * nblkbox;
                const int ncell = nviews * nsamp;
                // magic multipliers for the index decompositions below: lane i computes one, everybody fetches it
                uint32_t mg = 0u;
                if (lane < 5) mg = magic_of((uint32_t)(lane == 0 ? nblkbox : lane == 1 ? nbw : lane == 2 ? nsamp : lane == 3 ? ns : nu));
                const uint32_t m_nblkbox = __shfl_sync(FULL, mg, 0), m_nbw = __shfl_sync(FULL, mg, 1), m_nsamp = __shfl_sync(FULL, mg, 2),
                               m_ns = __shfl_sync(FULL, mg, 3), m_nu = __shfl_sync(FULL, mg, 4);
                __syncwarp();  // the previous range's cell reads are complete
                if (lane < h) { ws.lvl_base[lane] = incl - cntL; ws.lvl_pu0[lane] = pu0; ws.lvl_pv0[lane] = pv0; ws.lvl_nu[lane] = nuL; }
                // ------------------------------------------------------------ R: top-level RKV samples initialise the cells
                for (int q = lane; q < ncell; q += 32) {
                    const uint32_t vw = fdiv((uint32_t)q, m_nsamp), samp = (uint32_t)q - vw * (uint32_t)nsamp;
                    const uint32_t iv = fdiv(vw, m_nu), iu = vw - iv * (uint32_t)nu;
                    const uint32_t it = fdiv(samp, m_ns), is = samp - it * (uint32_t)ns;
                    const uint32_t top = (uint32_t)(((bv0 + (int)iv) >> h) * S.UH + ((bu0 + (int)iu) >> h));
                    const short4 rk = ldg(S.rkv + ((size_t)top * (size_t)S.Ht + (size_t)(bt0 + (int)it)) * (size_t)S.Ws + (size_t)(bs0 + (int)is));
                    ws.cell.acc[q] = make_int4(rk.x, rk.y, rk.z, 0);
                }
                __syncwarp();
                // ------------------------------------------------------------ S (part 2): slot table
                for (int s = lane; s < nslots; s += 32) {
                    int L = 0;
                    while (L + 1 < h && s >= ws.lvl_base[L + 1]) ++L;
                    const int jj = s - ws.lvl_base[L], n = ws.lvl_nu[L];
                    const int jv = jj / n;
                    const int pv = ws.lvl_pv0[L] + jv, pu = ws.lvl_pu0[L] + (jj - jv * n);
                    const LevelDesc lv = S.lev[L];
                    // views of the box below this plane: [iu0, iu1] x [iv0, iv1] relative to (bu0, bv0)
                    const int iu0 = max(pu << L, bu0) - bu0, iu1 = min(((pu + 1) << L) - 1, bu0 + nu - 1) - bu0;
                    const int iv0 = max(pv << L, bv0) - bv0, iv1 = min(((pv + 1) << L) - 1, bv0 + nv - 1) - bv0;
                    ws.slotinfo[s] = make_uint4(lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u,
                                                lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u, (uint32_t)((pu | pv) & 1),
                                                (uint32_t)(iu0 | (iu1 << 3) | (iv0 << 6) | (iv1 << 9)));
                }
                __syncwarp();

                // ------------------------------------------------------------ B1..B3, in chunks that fit the record / task queues
                const int s1 = bs0 + ns - 1, t1 = bt0 + nt - 1;
                const int rec_step = min(32, kTaskCap >> (2 * logB));  // records whose tasks always fit one B2 step
                                int *acc32 = reinterpret_cast<int *>(ws.cell.acc);
                int item_base = 0;
                while (item_base < nitems) {
                    // -------------------------------------------------------- B1: classify (plane, channel, block) items
                    int n_rec = 0;
                    while (item_base < nitems && n_rec + 32 <= kRecCap) {
                        const int it = item_base + lane;
                        bool keep = false;
                        uint4 r0, r1;
                        if (it < nitems) {
                            const uint32_t sc = fdiv((uint32_t)it, m_nblkbox), blk = (uint32_t)it - sc * (uint32_t)nblkbox;
                            const uint32_t slot = sc / 3u, c = sc - 3u * slot;
                            const uint32_t jb = fdiv(blk, m_nbw), ib = blk - jb * (uint32_t)nbw;
                            const uint4 si = ws.slotinfo[slot];
                            const uint4 d = ldg(S.pc + si.x + c);
                            const int b = (by0 + (int)jb) * S.nbx + bx0 + (int)ib;
                            const uint4 fr = ldg(S.flagrec + flag_index(S, si.x + (uint32_t)c, (uint32_t)(b >> 5)));  // = d.x + ..., without waiting for d
                            const uint32_t bit = 1u << (b & 31);
                            const bool res = (fr.x & bit) != 0u, pred = si.z && (fr.z & bit);
                            keep = res || pred;
                            // own payload base, rank * B^2, descriptor word, rank of the motion record | MV string base, reference pc, -, position
                            r0 = make_uint4(d.y, res ? ((fr.y + popc(fr.x & (bit - 1u))) << (2 * logB)) : 0xFFFFFFFFu, d.w,
                                            pred ? (fr.w + popc(fr.z & (bit - 1u))) : 0xFFFFFFFFu);
                            r1 = make_uint4(d.z, si.y + c, 0u, ib | (jb << 5) | (c << 10) | (si.w << 12));
                        }
                        const uint32_t bal = __ballot_sync(FULL, keep);
                        if (keep) {
                            const int idx = n_rec + (int)popc(bal & ((1u << lane) - 1u));
                            ws.q.rec[idx][0] = r0; ws.q.rec[idx][1] = r1;
                        }
                        n_rec += (int)popc(bal);
                        item_base += 32;
                    }
                    __syncwarp();
                    int rec_base = 0;
                    while (rec_base < n_rec) {
                        // ---------------------------------------------------- B2: motion record + reference descriptor once per block, emit value tasks
                        int n_task = 0;
                        while (rec_base < n_rec && n_task + (rec_step << (2 * logB)) <= kTaskCap) {
                            const int rr = rec_base + lane;
                            int cnt = 0, kxa = 0, kxb = -1, kya = 0, kyb = -1;
                            if (lane < rec_step && rr < n_rec) {
                                const uint4 r0 = ws.q.rec[rr][0], r1 = ws.q.rec[rr][1];
                                if (r0.w != 0xFFFFFFFFu) {
                                    const uint32_t rec = bise_at(S.mv + r1.x, r0.w, S.mv_layout, S.mv_m, lut);
                                    int md, dx, dy;
                                    mv_unpack(S, rec, md, dx, dy);
                                    const uint4 d = ldg(S.pc + r1.y);
                                    ws.q.rec[rr][0].w = 0x80000000u | ((uint32_t)md << 16) | ((uint32_t)(dx + S.W) << 8) | (uint32_t)(dy + S.W);
                                    ws.q.rec[rr][1] = make_uint4(d.x, d.y, d.w, r1.w);
                                } else {
                                    ws.q.rec[rr][0].w = 0u;
                                    ws.q.rec[rr][1] = make_uint4(0u, 0u, 0u, r1.w);  // B3 reads through these unconditionally
                                }
                                const int bx_ = (bx0 + (int)(r1.w & 31u)) << logB, by_ = (by0 + (int)((r1.w >> 5) & 31u)) << logB;
                                kxa = max(bx_, bs0) - bx_; kxb = min(bx_ + Bm1, s1) - bx_;
                                kya = max(by_, bt0) - by_; kyb = min(by_ + Bm1, t1) - by_;
                                cnt = (kxb - kxa + 1) * (kyb - kya + 1);
                            }
                            int inc = cnt;  // warp-inclusive scan: the records' tasks stay contiguous (coherent lanes in B3)
#pragma unroll
                            for (int o = 1; o < 32; o <<= 1) {
                                const int n = __shfl_up_sync(FULL, inc, o);
                                if (lane >= o) inc += n;
                            }
                            int o = n_task + inc - cnt;
                            n_task += __shfl_sync(FULL, inc, 31);
                            for (int ky = kya; ky <= kyb; ++ky)
                                for (int kx = kxa; kx <= kxb; ++kx) ws.q.task[o++] = (uint16_t)((rr << 6) | ((ky << logB) + kx));
                            rec_base += rec_step;
                        }
                        __syncwarp();
                        // ---------------------------------------------------- B3: one stored / re-compensated value per task
                        for (int t = lane; t < n_task; t += 32) {
                            const uint32_t task = ws.q.task[t];
                            const uint32_t rr = task >> 6, kin = task & 63u;
                            const uint4 r0 = ws.q.rec[rr][0], r1 = ws.q.rec[rr][1];
                            const int xx = ((bx0 + (int)(r1.w & 31u)) << logB) + (int)(kin & (uint32_t)Bm1);
                            const int yy = ((by0 + (int)((r1.w >> 5) & 31u)) << logB) + (int)(kin >> logB);
                            // straight-line: both decodes issue their loads at once (clamped / zero addresses where unused)
                            const bool own = r0.y != 0xFFFFFFFFu, pred = r0.w != 0u;
                            const int rx = xx + (int)((r0.w >> 8) & 0xFFu) - S.W, ryy = yy + (int)(r0.w & 0xFFu) - S.W;
                            const bool inb = pred && (unsigned)rx < (unsigned)S.Ws && (unsigned)ryy < (unsigned)S.Ht;
                            const int rxc = inb ? rx : 0, ryc = inb ? ryy : 0;
                            const int b = (ryc >> logB) * S.nbx + (rxc >> logB);
                            const uint4 fr = ldg(S.flagrec + r1.x + 4u * (uint32_t)(b >> 5));
                            const uint32_t vown = bise_at_uniform(S.pay + (own ? r0.x : 0u), own ? r0.y + kin : 0u, pc_layout(r0.z), pc_m(r0.z), lut);
                            const uint32_t bit = 1u << (b & 31);
                            const bool hasq = inb && (fr.x & bit) != 0u;
                            const uint32_t ii = ((fr.y + popc(fr.x & (bit - 1u))) << (2 * logB)) + (uint32_t)(((ryc & Bm1) << logB) + (rxc & Bm1));
                            const uint32_t vref = bise_at_uniform(S.pay + (hasq ? r1.y : 0u), hasq ? ii : 0u, pc_layout(r1.z), pc_m(r1.z), lut);
                            const int q = hasq ? pc_offset(r1.z) + (int)vref : 0;
                            // R10: subtractive P = e + R, additive P = e - R
                            const int e = (own ? pc_offset(r0.z) + (int)vown : 0) + ((r0.w & 0x10000u) ? -q : q);
                            if (e != 0) {
                                const int samp = (yy - bt0) * ns + (xx - bs0);
                                const int c = (int)((r1.w >> 10) & 3u);
                                const int iu0 = (int)((r1.w >> 12) & 7u), iu1 = (int)((r1.w >> 15) & 7u);
                                const int iv0 = (int)((r1.w >> 18) & 7u), iv1 = (int)((r1.w >> 21) & 7u);
                                if (iu0 == iu1 && iv0 == iv1) {  // one view below the plane (always so at level 0)
                                    atomicAdd(&acc32[(((iv0 * nu + iu0) * nsamp + samp) << 2) + c], e);
                                } else {
#pragma unroll 1
                                    for (int iv = iv0; iv <= iv1; ++iv)
#pragma unroll 1
                                        for (int iu = iu0; iu <= iu1; ++iu) atomicAdd(&acc32[(((iv * nu + iu) * nsamp + samp) << 2) + c], e);
                                }
                            }
                        }
                        __syncwarp();
                    }
                }
                {
                    // -------------------------------------------------------- B4: inverse colour transform, in place -> float RGB
                    for (int q = lane; q < ncell; q += 32) {
                        const int4 w = ws.cell.acc[q];
                        const int a[3] = {w.x, w.y, w.z};
                        const uint32_t c8 = ycocg_to_rgb8(a);
                        ws.cell.rgb[q] = make_float4((float)(c8 & 0xFFu), (float)((c8 >> 8) & 0xFFu), (float)((c8 >> 16) & 0xFFu), 0.f);
                    }
                    __syncwarp();

                    // -------------------------------------------------------- C: gather + blend
                    if (inr) {
#pragma unroll
                        for (int p = 0; p < kPPL; ++p)
                            if (pt[p].uv != 0xFFFFFFFFu) {
                                const int iu = (int)(pt[p].uv & 0xFFF) - bu0, iv = (int)((pt[p].uv >> 12) & 0xFFF) - bv0;
                                const int is = (int)(pt[p].st & 0x3FFF) - bs0, it = (int)((pt[p].st >> 14) & 0x3FFF) - bt0;
                                const int base = (iv * nu + iu) * nsamp + it * ns + is;
                                const int du = ((pt[p].uv >> 24) & 1u) ? nsamp : 0, dv = ((pt[p].uv >> 25) & 1u) ? nu * nsamp : 0;
                                const int ds = (int)((pt[p].st >> 28) & 1u), dt = ((pt[p].st >> 29) & 1u) ? ns : 0;
                                const float4 *patch = ws.cell.rgb;
                                rgb[p] = blend16(pt[p], [&](int a, int b) {
                                    return patch[base + ((a & 1) ? du : 0) + ((a & 2) ? dv : 0) + ((b & 1) ? ds : 0) + ((b & 2) ? dt : 0)];
                                });
                            }
                    }
                    done = true;
                }
            }
            if (!done) {
                if (span > 1) { span >>= 1; continue; }  // halve the range and try again
                // ---------------------------------------------------------------- single row still too large: 16 direct sample decodes
                if (inr) {
#pragma unroll
                    for (int p = 0; p < kPPL; ++p)
                        if (pt[p].uv != 0xFFFFFFFFu) rgb[p] = direct_pixel(S, pt[p]);
                }
            }
        }
        row0 += span;
        span = row0 & -row0;  // the largest aligned range that starts at row0 (row0 < 32 whenever it is used)
    }

    // ---------------------------------------------------------------- store: 3 kPPL contiguous bytes per lane
    if (y < H && x0 < W) {
        uint8_t *o = out + 3 * (((size_t)view * H + (size_t)y) * (size_t)W + (size_t)x0);
        if (kPPL % 4 == 0 && out_aligned && x0 + kPPL <= W) {
            uint32_t *o32 = reinterpret_cast<uint32_t *>(o);
#pragma unroll
            for (int g = 0; g < kPPL / 4; ++g) {
                o32[3 * g + 0] = rgb[4 * g] | (rgb[4 * g + 1] << 24);
                o32[3 * g + 1] = (rgb[4 * g + 1] >> 8) | (rgb[4 * g + 2] << 16);
                o32[3 * g + 2] = (rgb[4 * g + 2] >> 16) | (rgb[4 * g + 3] << 8);
            }
        } else if (kPPL == 2 && out_aligned && x0 + 2 <= W) {  // 6 bytes at an even offset: three 16-bit stores
            uint16_t *o16 = reinterpret_cast<uint16_t *>(o);
            o16[0] = (uint16_t)(rgb[0] & 0xFFFFu);
            o16[1] = (uint16_t)((rgb[0] >> 16) | ((rgb[1] & 0xFFu) << 8));
            o16[2] = (uint16_t)(rgb[1 % kPPL] >> 8);
        } else {
#pragma unroll
            for (int p = 0; p < kPPL; ++p)
                if (x0 + p < W) {
                    o[3 * p + 0] = (uint8_t)(rgb[p] & 0xFF);
                    o[3 * p + 1] = (uint8_t)((rgb[p] >> 8) & 0xFF);
                    o[3 * p + 2] = (uint8_t)((rgb[p] >> 16) & 0xFF);
                }
        }
    }
}

// (pixels per lane, warps per CTA, records, tasks, cells, min CTAs per SM)
using CfgA = Cfg<4, 4, 64, 512, 320, 6>;    // 16 x 8 tiles
using CfgB = Cfg<2, 4, 64, 512, 256, 7>;    // 8 x 8 tiles

template <class C>
cudaError_t launch_shape(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, cudaStream_t st)
{
    const int tiles_x = (W + C::kTileW - 1) / C::kTileW, tiles_y = (H + kTileH - 1) / kTileH;
    const long long tiles = (long long)tiles_x * tiles_y;
    if (tiles > 0x7fffffffLL) return cudaErrorInvalidValue;
    dim3 block(C::kWarps * 32), grid((unsigned)((tiles + C::kWarps - 1) / C::kWarps), (unsigned)n_views);
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0 && (W % 4) == 0) ? 1 : 0;
    render_warp_kernel<C><<<grid, block, C::kWarps * sizeof(WarpWs<C>), st>>>(S, d_cams, W, H, d_out, aligned, tiles_x, (int)tiles);
    return cudaGetLastError();
}

template <class C>
cudaError_t configure_shape()
{
    return cudaFuncSetAttribute(render_warp_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(C::kWarps * sizeof(WarpWs<C>)));
}

}  // namespace

cudaError_t configure_render_warp()
{
    cudaError_t e = configure_shape<CfgA>();
    if (e == cudaSuccess) e = configure_shape<CfgB>();
    return e;
}

cudaError_t launch_render_warp(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, cudaStream_t st,
                               int *n_launches, int shape)
{
    if (n_views == 0) return cudaSuccess;
    cudaError_t e = shape == 1 ? launch_shape<CfgB>(S, d_cams, n_views, W, H, d_out, st)
                                      : launch_shape<CfgA>(S, d_cams, n_views, W, H, d_out, st);
    if (n_launches) *n_launches += 1;
    return e;
}

}  // namespace hmlfc
