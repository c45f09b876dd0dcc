/* HMLFC oracle (test infrastructure) -- random-access decoder (paths P2 and P3) and the
 * algorithmic-bytes counter.
 *
 * PAPER.md:289-293 (section 4.8.1): "Decoding the blocks from the HMLFC hierarchy using tree
 * traversal; applying motion re-compensation for the motion compensated blocks.  At first,
 * the top-level RKV images are decoded and stored in memory. ... collect the required BISE
 * compressed SRV blocks from the top level to the bottom level.  Using the block indices,
 * we infer whether a block belongs to the predictive SRV images ... The motion vector values
 * for the corresponding block are decoded from the random accessible BISE compressed motion
 * vector stream.  The final pixel values are computed by combining the SRV pixel values
 * with the corresponding top-level RKV pixel values."
 * Pseudocode: SURVEY.md 8(c) C3 / DESIGN.md "Decoder".
 */
#include "oracle_internal.h"

#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static int flag_bit(const uint8_t *map, int b) { return (map[b >> 3] >> (b & 7)) & 1; }

static uint64_t pc_index(const orc_stream *s, int L, int pu, int pv, int c)
{
    return s->level_base[L] + ((uint64_t)pv * s->UL[L] + pu) * 3 + (uint64_t)c;
}

/* top-level RKV sample of channel c at (x,y) OF THAT CHANNEL'S PLANE: Y planes uint8, then the Co planes, then the Cg planes, int16 */
static int rkv_sample(const orc_stream *s, int c, int qu, int qv, int x, int y)
{
    const int h = s->h;
    const uint64_t n_top = (uint64_t)s->UL[h] * s->VL[h];
    const uint64_t npx = (uint64_t)s->g.W[c] * s->g.H[c];
    uint64_t i = ((uint64_t)qv * s->UL[h] + qu) * npx + (uint64_t)y * s->g.W[c] + x;
    const uint8_t *base = s->bytes + s->off_rkv;
    if (c == 0) return base[i];
    const uint8_t *q = base + n_top * (uint64_t)s->g.W[0] * s->g.H[0];
    if (c == 2) q += n_top * (uint64_t)s->g.W[1] * s->g.H[1] * 2;
    q += i * 2;
    return (int16_t)((uint16_t)q[0] | ((uint16_t)q[1] << 8));
}

/* stored value of plane-channel k at pixel (x,y) of its plane (channel k % 3): 0 if the block's res flag is clear.
 * use_rank = 1: rank directory + O(1) BISE addressing (P2).
 * use_rank = 0: linear scan of the flag map + sequential BISE decode (P3 brute force). */
static int plane_value(const orc_stream *s, uint64_t k, int x, int y, int use_rank)
{
    const int B = s->p.block;
    const orc_dirent *d = &s->dir[k];
    const uint8_t *fres = s->bytes + s->off_flags + d->flags_off;
    int b = (y / B) * s->g.nbx[k % 3] + (x / B);
    if (!flag_bit(fres, b)) return 0;
    const uint8_t *bits = s->bytes + s->off_payload + d->pay_bitoff / 8;
    int kk = (y % B) * B + (x % B);
    if (use_rank) {
        uint64_t i = (uint64_t)s->rank_res[k][b] * B * B + (uint64_t)kk;
        return d->offset + (int)orc_bise_decode_at(bits, d->N, i);
    }
    uint64_t rank = 0;
    for (int j = 0; j < b; ++j) rank += (uint64_t)flag_bit(fres, j);
    uint64_t i = rank * B * B + (uint64_t)kk;
    uint32_t *tmp = (uint32_t *)malloc((size_t)(i + 1) * sizeof(uint32_t));
    orc_bise_decode_seq(bits, d->N, i + 1, tmp);
    int v = d->offset + (int)tmp[i];
    free(tmp);
    return v;
}

/* stored sample of the reference plane k (channel c) at an integer position: 0 outside the image (R8) or in an insignificant block */
typedef struct { const orc_stream *s; uint64_t k; int c, use_rank; } ref_ctx;
static int ref_at(const void *ctx, int rx, int ry)
{
    const ref_ctx *r = (const ref_ctx *)ctx;
    if (rx < 0 || rx >= r->s->g.W[r->c] || ry < 0 || ry >= r->s->g.H[r->c]) return 0;
    return plane_value(r->s, r->k, rx, ry, r->use_rank);
}

static void decode_pixel(const orc_stream *s, int u, int v, int x, int y, int use_rank, uint8_t rgb[3])
{
    const int B = s->p.block, h = s->h;
    const int x0 = x, y0 = y;
    int acc[3];
    for (int c = 0; c < 3; ++c) {
        /* the channel's sample of light-field pixel (x0, y0): with chroma subsampling (R18) Co / Cg live at half resolution */
        const int x = x0 >> s->g.shift[c], y = y0 >> s->g.shift[c];
        const uint32_t fwords = (uint32_t)((s->g.nblk[c] + 31) / 32);
        int a = rkv_sample(s, c, u >> h, v >> h, x, y);
        for (int L = h - 1; L >= s->min_level; --L) { /* "from the top level to the bottom level"; progressive: stop early (R26) */
            int pu = u >> L, pv = v >> L;
            uint64_t k = pc_index(s, L, pu, pv, c);
            int e = plane_value(s, k, x, y, use_rank);
            if (orc_is_predictive(pu, pv)) {
                const orc_dirent *d = &s->dir[k];
                const uint8_t *fpred = s->bytes + s->off_flags + d->flags_off + (size_t)fwords * 4;
                int b = (y / B) * s->g.nbx[c] + (x / B);
                if (flag_bit(fpred, b)) {
                    uint64_t mi;
                    if (use_rank) mi = s->rank_pred[k][b];
                    else { mi = 0; for (int j = 0; j < b; ++j) mi += (uint64_t)flag_bit(fpred, j); }
                    const uint8_t *mbits = s->bytes + s->off_mv + d->mv_bitoff / 8;
                    uint32_t r;
                    if (use_rank) r = orc_bise_decode_at(mbits, s->mvN, mi);
                    else {
                        uint32_t *tmp = (uint32_t *)malloc((size_t)(mi + 1) * sizeof(uint32_t));
                        orc_bise_decode_seq(mbits, s->mvN, mi + 1, tmp);
                        r = tmp[mi];
                        free(tmp);
                    }
                    const int off = orc_mv_off(&s->p), nd = 2 * off + 1;
                    int mode = (int)(r / (uint32_t)(nd * nd));
                    int rem = (int)(r % (uint32_t)(nd * nd));
                    int dy = rem / nd - off, dx = rem % nd - off;
                    ref_ctx rc = {s, pc_index(s, L, pu & ~1, pv & ~1, c), c, use_rank};
                    /* R28: half-pel offsets read the bilinear mean of 1, 2 or 4 stored reference samples */
                    int q = s->p.subpel ? orc_halfpel(ref_at, &rc, 2 * x + dx, 2 * y + dy) : ref_at(&rc, x + dx, y + dy);
                    e += mode ? -q : q; /* R10: sub P = e + R, add P = e - R */
                }
            }
            a += e;
        }
        acc[c] = a;
    }
    int r, g, b;
    orc_ycocg_to_rgb(acc[0], acc[1], acc[2], &r, &g, &b);
    rgb[0] = (uint8_t)(r < 0 ? 0 : (r > 255 ? 255 : r));
    rgb[1] = (uint8_t)(g < 0 ? 0 : (g > 255 ? 255 : g));
    rgb[2] = (uint8_t)(b < 0 ? 0 : (b > 255 ? 255 : b));
}

int orc_set_min_level(orc_stream *s, int min_level)
{
    if (!s || min_level < 0 || min_level > s->h) return ORC_E_PARAM;
    s->min_level = min_level;
    return ORC_OK;
}

/* used by render.c */
void orc__decode_pixel(const orc_stream *s, int u, int v, int x, int y, uint8_t rgb[3])
{
    decode_pixel(s, u, v, x, y, 1, rgb);
}

static int in_range(const orc_stream *s, const int32_t *q)
{
    return q[0] >= 0 && q[0] < s->p.U && q[1] >= 0 && q[1] < s->p.V && q[2] >= 0 && q[2] < s->p.Ws && q[3] >= 0 && q[3] < s->p.Ht;
}

int64_t orc_decode(const orc_stream *s, const int32_t *coords, int64_t n, uint8_t *out, int nthreads)
{
    if (!s || !coords || !out || n < 0) return ORC_E_PARAM;
    int64_t oob = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(static) num_threads(nthreads) reduction(+ : oob)
    for (int64_t i = 0; i < n; ++i) {
        const int32_t *q = coords + 4 * i;
        if (!in_range(s, q)) { out[3 * i] = out[3 * i + 1] = out[3 * i + 2] = 0; ++oob; continue; }
        decode_pixel(s, q[0], q[1], q[2], q[3], 1, out + 3 * i);
    }
    return oob;
}

int64_t orc_decode_brute(const orc_stream *s, const int32_t *coords, int64_t n, uint8_t *out)
{
    if (!s || !coords || !out || n < 0) return ORC_E_PARAM;
    int64_t oob = 0;
    for (int64_t i = 0; i < n; ++i) {
        const int32_t *q = coords + 4 * i;
        if (!in_range(s, q)) { out[3 * i] = out[3 * i + 1] = out[3 * i + 2] = 0; ++oob; continue; }
        decode_pixel(s, q[0], q[1], q[2], q[3], 0, out + 3 * i);
    }
    return oob;
}

int orc_decode_full(const orc_stream *s, uint8_t *lf_out, int nthreads)
{
    if (!s || !lf_out) return ORC_E_PARAM;
    const int U = s->p.U, V = s->p.V, Ws = s->p.Ws, Ht = s->p.Ht;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(static) num_threads(nthreads)
    for (int64_t row = 0; row < (int64_t)U * V * Ht; ++row) {
        int y = (int)(row % Ht);
        int vi = (int)(row / Ht);
        int u = vi % U, v = vi / U;
        for (int x = 0; x < Ws; ++x) decode_pixel(s, u, v, x, y, 1, lf_out + ((size_t)row * Ws + x) * 3);
    }
    return ORC_OK;
}

/* ---------------------------------------------------------------- algorithmic bytes
 * every distinct (plane-channel, block) touched -- including reference
 * blocks reached through motion vectors -- counts once: its flag bits, its payload bits if
 * res, its motion record bits if pred; plus distinct top-RKV samples, output and input bytes.
 */
typedef struct {
    const orc_stream *s;
    uint8_t *blk_seen;  /* [n_pc * nblk of channel 0] */
    uint8_t *rkv_seen;  /* [3][n_top][npx of channel 0] */
    orc_stats st;
} stat_ctx;

/* bits per value in units of 1/15 bit (15 = lcm(3,5): whole groups in every layout) */
static int64_t bits15_per_value(uint32_t N) { return (int64_t)orc_bise_nbits(N, 15); }

static void touch_block(stat_ctx *cx, uint64_t k, int b, int is_pred_plane)
{
    const orc_stream *s = cx->s;
    uint8_t *seen = &cx->blk_seen[k * (uint64_t)s->g.nblk[0] + (uint64_t)b];
    if (*seen) return;
    *seen = 1;
    const orc_dirent *d = &s->dir[k];
    const uint32_t fwords = (uint32_t)((s->g.nblk[k % 3] + 31) / 32);
    const uint8_t *fres = s->bytes + s->off_flags + d->flags_off;
    cx->st.blocks_touched += 1;
    cx->st.flag_bits += is_pred_plane ? 2 : 1;
    if (flag_bit(fres, b)) cx->st.payload_bits15 += bits15_per_value(d->N) * s->p.block * s->p.block;
    if (is_pred_plane && flag_bit(fres + (size_t)fwords * 4, b)) cx->st.mv_bits15 += bits15_per_value(s->mvN);
}

static void touch_pixel(stat_ctx *cx, int u, int v, int x, int y)
{
    const orc_stream *s = cx->s;
    const int B = s->p.block, h = s->h;
    const uint64_t npx = (uint64_t)s->p.Ws * s->p.Ht, n_top = (uint64_t)s->UL[h] * s->VL[h];
    const int x0 = x, y0 = y;
    cx->st.taps += 1;
    for (int c = 0; c < 3; ++c) {
        const int x = x0 >> s->g.shift[c], y = y0 >> s->g.shift[c];  /* the channel's own sample (R18) */
        const uint32_t fwords = (uint32_t)((s->g.nblk[c] + 31) / 32);
        uint64_t ri = ((uint64_t)c * n_top + (uint64_t)(v >> h) * s->UL[h] + (u >> h)) * npx + (uint64_t)y * s->g.W[c] + x;
        if (!cx->rkv_seen[ri]) { cx->rkv_seen[ri] = 1; cx->st.rkv_bytes += (c == 0) ? 1 : 2; }
        for (int L = s->min_level; L < h; ++L) {
            int pu = u >> L, pv = v >> L;
            uint64_t k = pc_index(s, L, pu, pv, c);
            int b = (y / B) * s->g.nbx[c] + (x / B);
            int isp = orc_is_predictive(pu, pv);
            touch_block(cx, k, b, isp);
            if (!isp) continue;
            const orc_dirent *d = &s->dir[k];
            const uint8_t *fpred = s->bytes + s->off_flags + d->flags_off + (size_t)fwords * 4;
            if (!flag_bit(fpred, b)) continue;
            uint32_t r = orc_bise_decode_at(s->bytes + s->off_mv + d->mv_bitoff / 8, s->mvN, s->rank_pred[k][b]);
            const int off = orc_mv_off(&s->p), nd = 2 * off + 1;
            int rem = (int)(r % (uint32_t)(nd * nd));
            const int dx = rem % nd - off, dy = rem / nd - off;
            /* the integer samples the reference value is made of: one, or the 2 / 4 around a half-pel position (R28) */
            const int x2 = s->p.subpel ? 2 * x + dx : 2 * (x + dx), y2 = s->p.subpel ? 2 * y + dy : 2 * (y + dy);
            const int rx0 = orc_floor_div(x2, 2), ry0 = orc_floor_div(y2, 2);
            for (int jy = 0; jy <= (y2 - 2 * ry0); ++jy)
                for (int jx = 0; jx <= (x2 - 2 * rx0); ++jx) {
                    const int rx = rx0 + jx, ry = ry0 + jy;
                    if (rx >= 0 && rx < s->g.W[c] && ry >= 0 && ry < s->g.H[c])
                        touch_block(cx, pc_index(s, L, pu & ~1, pv & ~1, c), (ry / B) * s->g.nbx[c] + (rx / B), 0);
                }
        }
    }
}

static int stat_begin(stat_ctx *cx, const orc_stream *s)
{
    memset(cx, 0, sizeof(*cx));
    cx->s = s;
    uint64_t npx = (uint64_t)s->p.Ws * s->p.Ht, n_top = (uint64_t)s->UL[s->h] * s->VL[s->h];
    cx->blk_seen = (uint8_t *)calloc((size_t)(s->n_pc * (uint64_t)s->g.nblk[0]), 1);
    cx->rkv_seen = (uint8_t *)calloc((size_t)(3 * n_top * npx), 1);
    if (!cx->blk_seen || !cx->rkv_seen) { free(cx->blk_seen); free(cx->rkv_seen); return ORC_E_NOMEM; }
    return ORC_OK;
}

static void stat_end(stat_ctx *cx, orc_stats *out)
{
    cx->st.bytes_alg = ((double)cx->st.flag_bits + (double)(cx->st.payload_bits15 + cx->st.mv_bits15) / 15.0) / 8.0 + (double)cx->st.rkv_bytes +
                       (double)cx->st.out_bytes + (double)cx->st.in_bytes;
    *out = cx->st;
    free(cx->blk_seen);
    free(cx->rkv_seen);
}

int orc_stats_decode(const orc_stream *s, const int32_t *coords, int64_t n, orc_stats *out)
{
    if (!s || !coords || !out || n < 0) return ORC_E_PARAM;
    stat_ctx cx;
    int rc = stat_begin(&cx, s);
    if (rc) return rc;
    for (int64_t i = 0; i < n; ++i) {
        const int32_t *q = coords + 4 * i;
        if (in_range(s, q)) touch_pixel(&cx, q[0], q[1], q[2], q[3]);
    }
    cx.st.out_bytes = n * 3;
    cx.st.in_bytes = n * 16;
    stat_end(&cx, out);
    return ORC_OK;
}

/* implemented in render.c: enumerates the 16 taps of every hit pixel */
int orc__render_taps(const orc_stream *s, const float *cams, int n_views, int W, int H,
                     void (*cb)(void *, int, int, int, int), void *ud);

static void stat_tap_cb(void *ud, int u, int v, int x, int y) { touch_pixel((stat_ctx *)ud, u, v, x, y); }

int orc_stats_render(const orc_stream *s, const float *cams, int n_views, int W, int H, orc_stats *out)
{
    if (!s || !cams || !out || n_views < 0 || W <= 0 || H <= 0) return ORC_E_PARAM;
    stat_ctx cx;
    int rc = stat_begin(&cx, s);
    if (rc) return rc;
    orc__render_taps(s, cams, n_views, W, H, stat_tap_cb, &cx);
    cx.st.out_bytes = (int64_t)n_views * W * H * 3;
    cx.st.in_bytes = (int64_t)n_views * 64;
    stat_end(&cx, out);
    return ORC_OK;
}
