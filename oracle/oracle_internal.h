/* HMLFC oracle (test infrastructure) -- internal types shared by the oracle's own .c files only. */
#ifndef HMLFC_ORACLE_INTERNAL_H
#define HMLFC_ORACLE_INTERNAL_H

#include "hmlfc_oracle.h"

#define ORC_MAX_LEVELS 8

/* per-block record of a plane-channel */
typedef struct {
    int32_t mode;  /* 0 subtractive (P = e + R), 1 additive (P = e - R)  -- reading R10 */
    int32_t dx, dy;
    int32_t sad;   /* Delta = min(Delta-, Delta+) */
    int32_t E;     /* energy of the original SRV block: sum |px| */
    int32_t flags; /* bit0 res, bit1 pred */
} orc_block;

/* Per-channel plane geometry.  PAPER.md:263: "the chroma channels are sub-sampled ... The hierarchy computation and motion
 * compensation are performed separately on all the channels".  Reading R18: with p.chroma = 1 the Co and Cg planes of every input view
 * are reduced to Ws/2 x Ht/2 by a 2 x 2 box mean rounded half away from zero right after the colour transform; every
 * later step (hierarchy, search, thresholds, BISE, flag maps) runs on each channel at its own resolution with the same B and W; the
 * decoder reads the chroma sample (s >> 1, t >> 1): nearest-neighbour replication back to full size.  Ws, Ht must be even and B must
 * divide Ws/2 and Ht/2.  p.chroma = 0: all three channels at Ws x Ht. */
typedef struct {
    int W[3], H[3];          /* plane size of channel c        */
    int nbx[3], nby[3], nblk[3];
    int shift[3];            /* sample (s,t) -> (s >> shift, t >> shift) */
} orc_geom;

int orc__geom(const orc_params *p, orc_geom *g);  /* ORC_E_PARAM when the sizes do not divide */

struct orc_tree {
    orc_params p;
    orc_geom g;
    int h;
    int UL[ORC_MAX_LEVELS + 1], VL[ORC_MAX_LEVELS + 1];
    /* X[c][L][pv*UL+pu] : int16 [g.H[c]*g.W[c]], L = 0..h ; srv[c][L][...] : L = 0..h-1 */
    int16_t **X[3][ORC_MAX_LEVELS + 1];
    int16_t **srv[3][ORC_MAX_LEVELS];
    orc_block *blk[3][ORC_MAX_LEVELS]; /* [UL*VL][g.nblk[c]] */
    int thresholded;
};

/* ---- stream constants ---- */
#define ORC_HEADER_BYTES 160
#define ORC_DIRENT_BYTES 48
#define ORC_VERSION 1

/* directory entry as parsed */
typedef struct {
    int32_t offset;      /* value bias: stored value = offset + BISE value */
    uint32_t N;
    uint32_t n_res, n_pred;
    uint64_t flags_off;  /* bytes from the flags section */
    uint64_t pay_bitoff; /* bits from the payload section */
    uint64_t mv_bitoff;  /* bits from the MV section */
    int32_t layout, m;
} orc_dirent;

struct orc_stream {
    orc_params p;
    orc_geom g;
    int h;
    int UL[ORC_MAX_LEVELS + 1], VL[ORC_MAX_LEVELS + 1];
    uint8_t *bytes;
    size_t len;
    uint64_t off_rkv, off_dir, off_flags, off_payload, off_mv, total;
    uint64_t n_pc;
    orc_dirent *dir;            /* [n_pc] in stream order */
    uint64_t level_base[ORC_MAX_LEVELS]; /* first directory index of level L */
    uint32_t **rank_res;        /* [n_pc][g.nblk[c]+1] exclusive prefix counts (built at open) */
    uint32_t **rank_pred;       /* same for pred maps (NULL for reference planes) */
    uint32_t mvN;               /* 2 (2W+1)^2 */
    int min_level;              /* progressive decoding (R26): the walk stops above this level; 0 = full quality */
};

static inline int orc_is_predictive(int pu, int pv) { return ((pu | pv) & 1) != 0; }

/* ---- half-pel motion compensation (section 6: "sub-pel motion compensation, i.e., sub-pixel level motion compensation
 * to search for a matching block using bi-linear interpolation methods"; reading R28).  With p.subpel = 1 the
 * motion offsets (dx, dy) of a block are counted in HALF pixels, range [-2W, 2W]^2.  The reference value at the half-pel position
 * (x2 / 2, y2 / 2) is the bilinear interpolation there: the mean of the 1, 2 or 4 integer samples around it, rounded half up
 * (floor((sum + n/2) / n)); a sample outside the image reads 0 (R8).  Even offsets are the integer-pel case. */
static inline int orc_floor_div(int a, int n)  /* n > 0 */
{
    int q = a / n;
    return (a % n != 0 && a < 0) ? q - 1 : q;
}
typedef int (*orc_sample_fn)(const void *ctx, int x, int y);  /* reference sample at an integer position, 0 outside the image */
static inline int orc_halfpel(orc_sample_fn at, const void *ctx, int x2, int y2)
{
    const int x0 = orc_floor_div(x2, 2), y0 = orc_floor_div(y2, 2);
    const int fx = x2 - 2 * x0, fy = y2 - 2 * y0;
    int s = at(ctx, x0, y0), n = 1;
    if (fx) { s += at(ctx, x0 + 1, y0); n = 2; }
    if (fy) { s += at(ctx, x0, y0 + 1); if (fx) s += at(ctx, x0 + 1, y0 + 1); n *= 2; }
    return n == 1 ? s : orc_floor_div(s + n / 2, n);
}
/* a dense int16 plane as the sample source */
typedef struct { const int16_t *R; int W, H; } orc_plane_src;
static inline int orc_plane_at(const void *ctx, int x, int y)
{
    const orc_plane_src *p = (const orc_plane_src *)ctx;
    return (x >= 0 && x < p->W && y >= 0 && y < p->H) ? p->R[(size_t)y * p->W + x] : 0;
}
/* motion-record alphabet (R16): offsets in [-off, off], nd = 2 off + 1 values per axis, off = W (integer-pel) or 2W (half-pel) */
static inline int orc_mv_off(const orc_params *p) { return p->subpel ? 2 * p->window : p->window; }

#endif
