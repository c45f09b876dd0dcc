/* HMLFC oracle (test infrastructure) -- compressed stream writer and parser.
 *
 * PAPER.md:276 (section 4.7): "The HMLFC tree is linearized using breadth-first search (BFS)
 * traversal indexing all the SRVs in the traversal order starting from the top of the tree.
 * The BISE compressed blocks of the SRV images in the tree are arranged in the same BFS
 * linearized order and appended to the compressed stream. ... we extend the application of
 * BISE to encode the motion vector values."
 *
 * Byte layout "Stream format v1" is specified in DESIGN.md; all fields little-endian.
 * Plane-channel order: L = h-1 .. 0 (top of the tree first), planes row-major (pv outer, pu
 * inner), channel innermost (Y, Co, Cg).
 */
#include "oracle_internal.h"

#include <stdlib.h>
#include <string.h>

int orc__stored_value(const orc_tree *t, int c, int L, int pu, int pv, int x, int y);

static void wr16(uint8_t *p, uint32_t v) { p[0] = (uint8_t)v; p[1] = (uint8_t)(v >> 8); }
static void wr32(uint8_t *p, uint32_t v) { for (int i = 0; i < 4; ++i) p[i] = (uint8_t)(v >> (8 * i)); }
static void wr64(uint8_t *p, uint64_t v) { for (int i = 0; i < 8; ++i) p[i] = (uint8_t)(v >> (8 * i)); }
static uint32_t rd16(const uint8_t *p) { return (uint32_t)p[0] | ((uint32_t)p[1] << 8); }
static uint32_t rd32(const uint8_t *p) { uint32_t v = 0; for (int i = 0; i < 4; ++i) v |= (uint32_t)p[i] << (8 * i); return v; }
static uint64_t rd64(const uint8_t *p) { uint64_t v = 0; for (int i = 0; i < 8; ++i) v |= (uint64_t)p[i] << (8 * i); return v; }
static void wrf(uint8_t *p, float f) { uint32_t u; memcpy(&u, &f, 4); wr32(p, u); }
static float rdf(const uint8_t *p) { uint32_t u = rd32(p); float f; memcpy(&f, &u, 4); return f; }
static uint64_t align8(uint64_t x) { return (x + 7) & ~(uint64_t)7; }

/* joint motion record (R16): r = mode nd^2 + (dy + off) nd + (dx + off), nd = 2 off + 1; off = W, or 2W with half-pel offsets (R28) */
static uint32_t mv_pack(int mode, int dx, int dy, int off)
{
    uint32_t nd = (uint32_t)(2 * off + 1);
    return (uint32_t)mode * nd * nd + (uint32_t)(dy + off) * nd + (uint32_t)(dx + off);
}

int64_t orc_tree_serialize(const orc_tree *t, uint8_t **out)
{
    if (!t || !out || !t->thresholded) return ORC_E_PARAM;
    const int Ws = t->p.Ws, Ht = t->p.Ht, B = t->p.block, W = t->p.window, h = t->h;
    const uint32_t mvN = 2u * (uint32_t)(2 * orc_mv_off(&t->p) + 1) * (uint32_t)(2 * orc_mv_off(&t->p) + 1);

    uint64_t n_pc = 0;
    for (int L = 0; L < h; ++L) n_pc += (uint64_t)t->UL[L] * t->VL[L] * 3;
    orc_dirent *dir = (orc_dirent *)calloc((size_t)n_pc, sizeof(orc_dirent));
    if (!dir) return ORC_E_NOMEM;

    /* pass 1: ranges and section sizes */
    uint64_t flags_bytes = 0, pay_bits = 0, mv_bits = 0, k = 0;
    for (int L = h - 1; L >= 0; --L)
        for (int pv = 0; pv < t->VL[L]; ++pv)
            for (int pu = 0; pu < t->UL[L]; ++pu)
                for (int c = 0; c < 3; ++c, ++k) {
                    const int nblk = t->g.nblk[c];  /* every channel at its own resolution (R18) */
                    const uint32_t fwords = (uint32_t)((nblk + 31) / 32);
                    const orc_block *bk = t->blk[c][L] + (size_t)(pv * t->UL[L] + pu) * nblk;
                    int vmin = 0, vmax = 0, first = 1;
                    uint32_t n_res = 0, n_pred = 0;
                    for (int b = 0; b < nblk; ++b) {
                        if (bk[b].flags & 2) ++n_pred;
                        if (!(bk[b].flags & 1)) continue;
                        ++n_res;
                        int bx = b % t->g.nbx[c], by = b / t->g.nbx[c];
                        for (int j = 0; j < B; ++j)
                            for (int i = 0; i < B; ++i) {
                                int v = orc__stored_value(t, c, L, pu, pv, bx * B + i, by * B + j);
                                if (first) { vmin = vmax = v; first = 0; }
                                if (v < vmin) vmin = v;
                                if (v > vmax) vmax = v;
                            }
                    }
                    orc_dirent *d = &dir[k];
                    d->offset = vmin;
                    d->N = (uint32_t)(vmax - vmin + 1);
                    d->n_res = n_res;
                    d->n_pred = n_pred;
                    orc_bise_choose(d->N, &d->layout, &d->m);
                    d->flags_off = flags_bytes;
                    flags_bytes += (uint64_t)fwords * 4 * (orc_is_predictive(pu, pv) ? 2 : 1);
                    d->pay_bitoff = pay_bits;
                    pay_bits += orc_bise_nbits(d->N, (uint64_t)n_res * B * B);
                    pay_bits = (pay_bits + 31) & ~(uint64_t)31;
                    d->mv_bitoff = mv_bits;
                    mv_bits += orc_bise_nbits(mvN, n_pred);
                    mv_bits = (mv_bits + 31) & ~(uint64_t)31;
                }

    uint64_t n_top = (uint64_t)t->UL[h] * t->VL[h];
    uint64_t rkv_bytes = 0;
    for (int c = 0; c < 3; ++c) rkv_bytes += n_top * (uint64_t)t->g.W[c] * t->g.H[c] * (c == 0 ? 1 : 2);
    uint64_t off_rkv = ORC_HEADER_BYTES;
    uint64_t off_dir = align8(off_rkv + rkv_bytes);
    uint64_t off_flags = align8(off_dir + n_pc * ORC_DIRENT_BYTES);
    uint64_t off_payload = align8(off_flags + flags_bytes);
    uint64_t off_mv = align8(off_payload + pay_bits / 8 + 8);
    uint64_t total = align8(off_mv + mv_bits / 8 + 8);

    uint8_t *s = (uint8_t *)calloc((size_t)total, 1);
    if (!s) { free(dir); return ORC_E_NOMEM; }

    /* header */
    memcpy(s, "HMLF", 4);
    wr16(s + 4, ORC_VERSION);
    wr16(s + 6, ORC_HEADER_BYTES);
    wr32(s + 8, (uint32_t)t->p.U); wr32(s + 12, (uint32_t)t->p.V); wr32(s + 16, (uint32_t)Ws); wr32(s + 20, (uint32_t)Ht);
    wr32(s + 24, (uint32_t)h); wr32(s + 28, (uint32_t)B); wr32(s + 32, (uint32_t)W); wr32(s + 36, 3);
    wr32(s + 40, (uint32_t)t->p.tau_ref); wr32(s + 44, (uint32_t)t->p.tau_res);
    s[48] = 1; /* colour id: YCoCg-R */
    s[49] = t->p.chroma ? 1 : 0; /* chroma subsampling (R18): Co / Cg planes at Ws/2 x Ht/2 */
    s[50] = 0; /* RKV codec: raw (R20) */
    s[51] = (uint8_t)t->p.policy;
    s[52] = t->p.background[0]; s[53] = t->p.background[1]; s[54] = t->p.background[2];
    s[55] = t->p.subpel ? 1 : 0; /* motion offsets in half pixels (R28) */
    wrf(s + 56, t->p.uv_origin[0]); wrf(s + 60, t->p.uv_origin[1]);
    wrf(s + 64, t->p.uv_step[0]);   wrf(s + 68, t->p.uv_step[1]);
    wrf(s + 72, t->p.st_origin[0]); wrf(s + 76, t->p.st_origin[1]);
    wrf(s + 80, t->p.st_step[0]);   wrf(s + 84, t->p.st_step[1]);
    wrf(s + 88, t->p.z_st);
    wr32(s + 92, 0);
    wr64(s + 96, t->p.seed);
    wr64(s + 104, n_pc);
    wr64(s + 112, off_rkv); wr64(s + 120, off_dir); wr64(s + 128, off_flags);
    wr64(s + 136, off_payload); wr64(s + 144, off_mv); wr64(s + 152, total);

    /* top-level RKVs, raw: channel-major; Y uint8, Co/Cg int16 LE (R6, R20) */
    {
        uint8_t *o = s + off_rkv;
        for (uint64_t i = 0; i < n_top; ++i)
            for (size_t x = 0; x < (size_t)t->g.W[0] * t->g.H[0]; ++x) *o++ = (uint8_t)t->X[0][h][i][x];
        for (int c = 1; c < 3; ++c)
            for (uint64_t i = 0; i < n_top; ++i)
                for (size_t x = 0; x < (size_t)t->g.W[c] * t->g.H[c]; ++x) { wr16(o, (uint32_t)(uint16_t)t->X[c][h][i][x]); o += 2; }
    }

    /* pass 2: directory, flag maps, payloads, motion vectors */
    uint32_t *vals = (uint32_t *)malloc((size_t)t->g.nblk[0] * B * B * sizeof(uint32_t));  /* channel 0 has the most blocks */
    uint32_t *mvs = (uint32_t *)malloc((size_t)t->g.nblk[0] * sizeof(uint32_t));
    if (!vals || !mvs) { free(vals); free(mvs); free(dir); free(s); return ORC_E_NOMEM; }
    k = 0;
    for (int L = h - 1; L >= 0; --L)
        for (int pv = 0; pv < t->VL[L]; ++pv)
            for (int pu = 0; pu < t->UL[L]; ++pu)
                for (int c = 0; c < 3; ++c, ++k) {
                    const orc_dirent *d = &dir[k];
                    const int nblk = t->g.nblk[c];
                    const uint32_t fwords = (uint32_t)((nblk + 31) / 32);
                    const orc_block *bk = t->blk[c][L] + (size_t)(pv * t->UL[L] + pu) * nblk;
                    int is_pred = orc_is_predictive(pu, pv);
                    uint8_t *e = s + off_dir + k * ORC_DIRENT_BYTES;
                    wr32(e, (uint32_t)d->offset); wr32(e + 4, d->N); wr32(e + 8, d->n_res); wr32(e + 12, d->n_pred);
                    wr64(e + 16, d->flags_off); wr64(e + 24, d->pay_bitoff); wr64(e + 32, d->mv_bitoff);
                    e[40] = (uint8_t)d->layout; e[41] = (uint8_t)d->m; e[42] = (uint8_t)is_pred; e[43] = 0;
                    wr32(e + 44, 0);
                    uint8_t *fres = s + off_flags + d->flags_off;
                    uint8_t *fpred = fres + (size_t)fwords * 4;
                    uint64_t nv = 0, nm = 0;
                    for (int b = 0; b < nblk; ++b) {
                        if (bk[b].flags & 2) {
                            fpred[b >> 3] |= (uint8_t)(1u << (b & 7));
                            mvs[nm++] = mv_pack(bk[b].mode, bk[b].dx, bk[b].dy, orc_mv_off(&t->p));
                        }
                        if (!(bk[b].flags & 1)) continue;
                        fres[b >> 3] |= (uint8_t)(1u << (b & 7));
                        int bx = b % t->g.nbx[c], by = b / t->g.nbx[c];
                        for (int j = 0; j < B; ++j)
                            for (int i = 0; i < B; ++i)
                                vals[nv++] = (uint32_t)(orc__stored_value(t, c, L, pu, pv, bx * B + i, by * B + j) - d->offset);
                    }
                    if (nv) orc_bise_encode(vals, nv, d->N, s + off_payload + d->pay_bitoff / 8);
                    if (nm) orc_bise_encode(mvs, nm, mvN, s + off_mv + d->mv_bitoff / 8);
                }
    free(vals);
    free(mvs);
    free(dir);
    *out = s;
    return (int64_t)total;
}

/* ---------------------------------------------------------------- parser */
void orc_close(orc_stream *s)
{
    if (!s) return;
    if (s->rank_res) for (uint64_t i = 0; i < s->n_pc; ++i) free(s->rank_res[i]);
    if (s->rank_pred) for (uint64_t i = 0; i < s->n_pc; ++i) free(s->rank_pred[i]);
    free(s->rank_res);
    free(s->rank_pred);
    free(s->dir);
    free(s->bytes);
    free(s);
}

orc_stream *orc_open(const uint8_t *bytes, size_t len, int *err)
{
    int e_dummy;
    if (!err) err = &e_dummy;
    *err = ORC_OK;
    if (!bytes || len < 8) { *err = ORC_E_TRUNCATED; return NULL; }
    if (memcmp(bytes, "HMLF", 4) != 0) { *err = ORC_E_MAGIC; return NULL; }
    if (rd16(bytes + 4) != ORC_VERSION) { *err = ORC_E_VERSION; return NULL; }
    if (len < ORC_HEADER_BYTES) { *err = ORC_E_TRUNCATED; return NULL; }
    orc_stream *s = (orc_stream *)calloc(1, sizeof(orc_stream));
    if (!s) { *err = ORC_E_NOMEM; return NULL; }
    s->p.U = (int32_t)rd32(bytes + 8); s->p.V = (int32_t)rd32(bytes + 12);
    s->p.Ws = (int32_t)rd32(bytes + 16); s->p.Ht = (int32_t)rd32(bytes + 20);
    s->p.height = (int32_t)rd32(bytes + 24); s->p.block = (int32_t)rd32(bytes + 28); s->p.window = (int32_t)rd32(bytes + 32);
    uint32_t nch = rd32(bytes + 36);
    s->p.tau_ref = (int32_t)rd32(bytes + 40); s->p.tau_res = (int32_t)rd32(bytes + 44);
    s->p.policy = bytes[51];
    s->p.background[0] = bytes[52]; s->p.background[1] = bytes[53]; s->p.background[2] = bytes[54];
    s->p.uv_origin[0] = rdf(bytes + 56); s->p.uv_origin[1] = rdf(bytes + 60);
    s->p.uv_step[0] = rdf(bytes + 64);   s->p.uv_step[1] = rdf(bytes + 68);
    s->p.st_origin[0] = rdf(bytes + 72); s->p.st_origin[1] = rdf(bytes + 76);
    s->p.st_step[0] = rdf(bytes + 80);   s->p.st_step[1] = rdf(bytes + 84);
    s->p.z_st = rdf(bytes + 88);
    s->p.seed = rd64(bytes + 96);
    s->n_pc = rd64(bytes + 104);
    s->off_rkv = rd64(bytes + 112); s->off_dir = rd64(bytes + 120); s->off_flags = rd64(bytes + 128);
    s->off_payload = rd64(bytes + 136); s->off_mv = rd64(bytes + 144); s->total = rd64(bytes + 152);
    const orc_params *p = &s->p;
    s->p.chroma = bytes[49];
    s->p.subpel = bytes[55];
    if (rd16(bytes + 6) != ORC_HEADER_BYTES || nch != 3 || bytes[48] != 1 || bytes[49] > 1 || bytes[50] != 0 || bytes[55] > 1 ||
        p->U < 1 || p->V < 1 || p->Ws < 1 || p->Ht < 1 || p->height < 1 || p->height > ORC_MAX_LEVELS || p->block < 1 ||
        p->block > 8 || p->window < 0 || p->window > 64 || orc__geom(p, &s->g) != ORC_OK) {
        free(s); *err = ORC_E_PARAM; return NULL;
    }
    if (len < s->total) { free(s); *err = ORC_E_TRUNCATED; return NULL; }
    s->h = p->height;
    uint64_t n_pc = 0;
    for (int L = 0; L <= s->h; ++L) {
        s->UL[L] = (p->U + (1 << L) - 1) >> L;
        s->VL[L] = (p->V + (1 << L) - 1) >> L;
    }
    for (int L = s->h - 1; L >= 0; --L) { s->level_base[L] = n_pc; n_pc += (uint64_t)s->UL[L] * s->VL[L] * 3; }
    uint64_t rkv_bytes = 0;
    for (int c = 0; c < 3; ++c) rkv_bytes += (uint64_t)s->UL[s->h] * s->VL[s->h] * (uint64_t)s->g.W[c] * s->g.H[c] * (c == 0 ? 1 : 2);
    if (n_pc != s->n_pc || s->off_rkv != ORC_HEADER_BYTES || s->off_dir < s->off_rkv + rkv_bytes ||
        s->off_flags < s->off_dir + n_pc * ORC_DIRENT_BYTES || s->off_payload < s->off_flags || s->off_mv < s->off_payload ||
        s->total < s->off_mv) {
        free(s); *err = ORC_E_CORRUPT; return NULL;
    }
    s->mvN = 2u * (uint32_t)(2 * orc_mv_off(p) + 1) * (uint32_t)(2 * orc_mv_off(p) + 1);
    s->len = (size_t)s->total;
    s->bytes = (uint8_t *)malloc(s->len);
    s->dir = (orc_dirent *)calloc((size_t)n_pc, sizeof(orc_dirent));
    s->rank_res = (uint32_t **)calloc((size_t)n_pc, sizeof(uint32_t *));
    s->rank_pred = (uint32_t **)calloc((size_t)n_pc, sizeof(uint32_t *));
    if (!s->bytes || !s->dir || !s->rank_res || !s->rank_pred) { orc_close(s); *err = ORC_E_NOMEM; return NULL; }
    memcpy(s->bytes, bytes, s->len);
    for (uint64_t k = 0; k < n_pc; ++k) {
        const int nblk = s->g.nblk[k % 3];  /* channel = k % 3 (level bases are multiples of 3) */
        const uint32_t fwords = (uint32_t)((nblk + 31) / 32);
        const uint8_t *e = s->bytes + s->off_dir + k * ORC_DIRENT_BYTES;
        orc_dirent *d = &s->dir[k];
        d->offset = (int32_t)rd32(e); d->N = rd32(e + 4); d->n_res = rd32(e + 8); d->n_pred = rd32(e + 12);
        d->flags_off = rd64(e + 16); d->pay_bitoff = rd64(e + 24); d->mv_bitoff = rd64(e + 32);
        d->layout = e[40]; d->m = e[41];
        int is_pred = e[42];
        int32_t lay, m;
        orc_bise_choose(d->N, &lay, &m);
        uint64_t fbytes = (uint64_t)fwords * 4 * (is_pred ? 2 : 1);
        if (lay != d->layout || m != d->m || d->N < 1 || s->off_flags + d->flags_off + fbytes > s->off_payload ||
            s->off_payload + (d->pay_bitoff + orc_bise_nbits(d->N, (uint64_t)d->n_res * p->block * p->block)) / 8 > s->off_mv ||
            s->off_mv + (d->mv_bitoff + orc_bise_nbits(s->mvN, d->n_pred)) / 8 > s->total) {
            orc_close(s); *err = ORC_E_CORRUPT; return NULL;
        }
        /* rank directory: exclusive prefix popcounts of the flag maps */
        const uint8_t *fres = s->bytes + s->off_flags + d->flags_off;
        uint32_t *rr = (uint32_t *)malloc((size_t)(nblk + 1) * sizeof(uint32_t));
        if (!rr) { orc_close(s); *err = ORC_E_NOMEM; return NULL; }
        s->rank_res[k] = rr;
        uint32_t acc = 0;
        for (int b = 0; b < nblk; ++b) { rr[b] = acc; acc += (fres[b >> 3] >> (b & 7)) & 1u; }
        rr[nblk] = acc;
        if (acc != d->n_res) { orc_close(s); *err = ORC_E_CORRUPT; return NULL; }
        if (is_pred) {
            const uint8_t *fpred = fres + (size_t)fwords * 4;
            uint32_t *rp = (uint32_t *)malloc((size_t)(nblk + 1) * sizeof(uint32_t));
            if (!rp) { orc_close(s); *err = ORC_E_NOMEM; return NULL; }
            s->rank_pred[k] = rp;
            acc = 0;
            for (int b = 0; b < nblk; ++b) { rp[b] = acc; acc += (fpred[b >> 3] >> (b & 7)) & 1u; }
            rp[nblk] = acc;
            if (acc != d->n_pred) { orc_close(s); *err = ORC_E_CORRUPT; return NULL; }
        } else if (d->n_pred != 0) { orc_close(s); *err = ORC_E_CORRUPT; return NULL; }
    }
    return s;
}

int orc_stream_params(const orc_stream *s, orc_params *out)
{
    if (!s || !out) return ORC_E_PARAM;
    *out = s->p;
    return ORC_OK;
}
