/*
 * HMLFC oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation of HMLFC (Pratapa & Manocha,
 * arXiv 1902.09396) written step by step from /root/reference/PAPER.md, following the
 * readings ledgered in DESIGN.md ("Readings of the paper", R1..R25).  It produces the
 * compressed streams the CUDA path consumes and the expected decoded pixels / rendered
 * views the CUDA path is compared against.
 *
 * Rules: only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this library.  It shares no code, header,
 * table or constant with paper_1902_09396_b200/csrc/ (the CUDA path) and neither includes
 * the other.  All arithmetic is integer (int16 storage, int32 accumulation) except the
 * renderer: ray set-up in strict IEEE fp32 (-ffp-contract=off), blend in fp64.
 *
 * Parity pins: every function is pinned by tests/test_oracle_*.py (-m "not gpu") against
 * closed forms, brute force, invariants or the paper's statements.  Unpinned: the paper's
 * Table 1/2 bpp/PSNR numbers ("parity unpinned": the Stanford light fields are not
 * available and the container / RKV codec differ).
 *
 * Notation: (u,v) camera-grid index, U x V views;
 * (s,t) pixel column/row, Ws x Ht.  Level L in [0,h-1] has U_L x V_L SRV planes,
 * U_L = ceil(U / 2^L); top RKVs are level h.  Level 0 is the finest.
 */
#ifndef HMLFC_ORACLE_H
#define HMLFC_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes (oracle's own numbering) ---- */
enum {
    ORC_OK = 0,
    ORC_E_MAGIC = -1,
    ORC_E_TRUNCATED = -2,
    ORC_E_VERSION = -3,
    ORC_E_PARAM = -4,
    ORC_E_NOMEM = -5,
    ORC_E_CORRUPT = -6
};

/* encoder policies for the per-block (pred,res) decision: DESIGN.md reading R13 */
/* ORC_POLICY_NOMOTION: no block is ever predicted -- the RLFC hierarchy without the motion compensation this paper adds (PAPER.md:183,
 * "RLFC"; :375 compares HMLFC against it).  Same stream format, same decoder: a stream without motion records. */
enum { ORC_POLICY_ADAPTIVE = 0, ORC_POLICY_ALL = 1, ORC_POLICY_LITERAL = 2, ORC_POLICY_NOMOTION = 3 };

/* BISE layouts (section 4.6) */
enum { ORC_BISE_PLAIN = 0, ORC_BISE_TRIT = 1, ORC_BISE_QUINT = 2 };

typedef struct {
    int32_t U, V, Ws, Ht;      /* light-field shape                                   */
    int32_t height;            /* tree height h ("tree height")          */
    int32_t block;             /* block size B ("block size")                          */
    int32_t window;            /* search window W ("search window size")               */
    int32_t tau_ref, tau_res;  /* the two block thresholds              */
    int32_t policy;            /* ORC_POLICY_*                                         */
    int32_t nthreads;          /* OpenMP threads (<=0: all)                            */
    float uv_origin[2], uv_step[2], st_origin[2], st_step[2], z_st; /* light slab      */
    uint8_t background[3];
    uint8_t chroma;            /* 1: Co / Cg at half resolution (R18)    */
    uint8_t subpel;            /* 1: half-pel motion compensation (R28)   */
    uint64_t seed;             /* provenance only                                      */
} orc_params;

/* ------------------------------------------------------------------ colour */
void orc_rgb_to_ycocg(int r, int g, int b, int *y, int *co, int *cg);
void orc_ycocg_to_rgb(int y, int co, int cg, int *r, int *g, int *b); /* no clamp */
/* exhaustive 2^24 round trip; returns the number of failing triples (pin) */
int64_t orc_colour_roundtrip_failures(void);

/* ------------------------------------------------------------------ BISE */
typedef struct {
    uint32_t N;        /* values in [0, N-1] */
    int32_t layout;    /* ORC_BISE_* */
    int32_t m;         /* low bits per value */
    uint64_t count;    /* number of values */
    uint64_t nbits;    /* payload length in bits (whole groups) */
} orc_bise_info;

void orc_bise_choose(uint32_t N, int32_t *layout, int32_t *m);
uint64_t orc_bise_nbits(uint32_t N, uint64_t count);
/* encode count values into bits (LSB-first bit string, caller provides >= nbits/8+8 zeroed bytes) */
int orc_bise_encode(const uint32_t *values, uint64_t count, uint32_t N, uint8_t *bits);
uint32_t orc_bise_decode_at(const uint8_t *bits, uint32_t N, uint64_t i);
/* sequential decode of the first count values (independent routine used by the P3 decoder) */
void orc_bise_decode_seq(const uint8_t *bits, uint32_t N, uint64_t count, uint32_t *out);

/* ------------------------------------------------------------------ encoder */
typedef struct orc_tree orc_tree;

/* colour transform + hierarchy + roles + exhaustive phase-shifted search; tau-independent */
orc_tree *orc_encode_begin(const uint8_t *lf /* [V][U][Ht][Ws][3] RGB8 */, const orc_params *p, int *err);
/* two-threshold significance + per-block (pred,res) decision */
int orc_tree_threshold(orc_tree *t, int tau_ref, int tau_res, int policy);
/* BFS linearisation + BISE + stream assembly; *out is malloc'ed (free with orc_free) */
int64_t orc_tree_serialize(const orc_tree *t, uint8_t **out);
/* P1: the encoder's own dense top-down reconstruction -> RGB8 [V][U][Ht][Ws][3] */
int orc_tree_reconstruct(const orc_tree *t, uint8_t *lf_out);
void orc_tree_free(orc_tree *t);
void orc_free(void *p);

/* introspection used by the pins */
int orc_tree_level_dims(const orc_tree *t, int L, int *UL, int *VL);
/* copy plane (L,pu,pv,channel): kind 0 = X_L (L in [0,h]), 1 = SRV_L (original, L<h),
 * 2 = stored values (reference: SRV; predictive: residual e incl. intra), int16 [Ht][Ws] */
int orc_tree_get_plane(const orc_tree *t, int kind, int L, int pu, int pv, int c, int16_t *out);
/* per-block records of plane (L,pu,pv,c): out[nblk][6] = mode,dx,dy,sad,E_P,flags(bit0 res, bit1 pred) */
int orc_tree_get_blocks(const orc_tree *t, int L, int pu, int pv, int c, int32_t *out);
/* search one block directly (pin): P,R int16 planes [Ht][Ws]; writes mode,dx,dy,sad */
void orc_search_block(const int16_t *P, const int16_t *R, int Ws, int Ht, int B, int W, int bx, int by,
                      int32_t out[4]);
/* the same on the half-pel grid (R28): out = {mode, dx2, dy2, Delta}, offsets in half pixels, range [-2W, 2W] */
void orc_search_block_halfpel(const int16_t *P, const int16_t *R, int Ws, int Ht, int B, int W, int bx, int by, int32_t out[4]);

/* ------------------------------------------------------------------ decoder */
typedef struct orc_stream orc_stream;

orc_stream *orc_open(const uint8_t *bytes, size_t len, int *err); /* copies bytes */
void orc_close(orc_stream *s);
/* Progressive decoding (PAPER.md:57, :183 name the property; :289-293 the top-down traversal it truncates; R26): the
 * decoder and the renderer sum the top-level RKV and the levels h-1 .. min_level only (0 = everything, h = the top RKV alone), which
 * yields the representative key view of the level-min_level cluster that contains the view.  Returns ORC_E_PARAM outside [0, h]. */
int orc_set_min_level(orc_stream *s, int min_level);
int orc_stream_params(const orc_stream *s, orc_params *out);
/* P2: per-pixel random access; coords [n][4] = u,v,s,t ; out [n][3] RGB8; out-of-range -> (0,0,0).
 * Returns the number of out-of-range coordinates. */
int64_t orc_decode(const orc_stream *s, const int32_t *coords, int64_t n, uint8_t *out, int nthreads);
/* P3: brute force (no rank directory use, sequential BISE decode); tiny inputs only */
int64_t orc_decode_brute(const orc_stream *s, const int32_t *coords, int64_t n, uint8_t *out);
/* whole light field via P2 */
int orc_decode_full(const orc_stream *s, uint8_t *lf_out, int nthreads);

/* ------------------------------------------------------------------ renderer */
/* camera: 16 floats = eye[3], right[3], down[3], fwd[3], tan_half_x, tan_half_y, pad[2] */
int orc_render(const orc_stream *s, const float *cams, int n_views, int W, int H, uint8_t *out, int nthreads);
/* per-view level of detail (R27): view k stops the walk above levels[k]; orc_lod_level = floor(log2(|z_st - eye.z| / d0)) in [0, h] */
int orc_render_lod(const orc_stream *s, const float *cams, const int32_t *levels, int n_views, int W, int H, uint8_t *out, int nthreads);
int orc_lod_level(const orc_params *p, const float *cam, float d0);
/* same sampling path, pixels taken from a dense RGB8 light field (pin: render-from-stream = render-from-LF) */
int orc_render_dense(const uint8_t *lf, const orc_params *p, const float *cams, int n_views, int W, int H,
                     uint8_t *out, int nthreads);
/* ray set-up only: out[W*H][5] = u,v,s,t (continuous), hit flag (1.0 / 0.0) */
int orc_ray_setup(const orc_params *p, const float *cam, int W, int H, float *out);

/* ------------------------------------------------------------------ stats / metrics */
typedef struct {
    int64_t taps;              /* tap decodes requested                                  */
    int64_t blocks_touched;    /* distinct (plane-channel, block) incl. reference blocks */
    int64_t flag_bits;         /* 1 (reference) or 2 (predictive) bits per distinct block */
    int64_t payload_bits15;    /* B^2 * bits/value for distinct res blocks, in 1/15 bit  */
    int64_t mv_bits15;         /* distinct pred blocks * bits/record, in 1/15 bit        */
    int64_t rkv_bytes;         /* distinct top-RKV samples * (1|2) bytes                 */
    int64_t out_bytes, in_bytes;
    double bytes_alg;          /* total                                  */
} orc_stats;
int orc_stats_decode(const orc_stream *s, const int32_t *coords, int64_t n, orc_stats *out);
int orc_stats_render(const orc_stream *s, const float *cams, int n_views, int W, int H, orc_stats *out);

double orc_psnr(const uint8_t *a, const uint8_t *b, int64_t n); /* 10 log10(255^2 / MSE) */

#ifdef __cplusplus
}
#endif
#endif
