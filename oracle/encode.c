/* HMLFC oracle (test infrastructure) -- encoder: colour, RLFC hierarchy, phase-shifted motion
 * compensation, thresholds, and the encoder's own dense reconstruction (decode path P1).
 *
 * Follows PAPER.md sections 4.3-4.5 in the paper's order; readings in DESIGN.md (R1..R13).
 */
#include "oracle_internal.h"

#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static int iabs(int x) { return x < 0 ? -x : x; }

/* round(sum / n), half away from zero, n in {1,2,4}  (reading R2: uniform mean filter) */
static int round_mean(int sum, int n)
{
    if (sum >= 0) return (2 * sum + n) / (2 * n);
    return -((-2 * sum + n) / (2 * n));
}

int orc__geom(const orc_params *p, orc_geom *g)
{
    if (p->block < 1) return ORC_E_PARAM;
    for (int c = 0; c < 3; ++c) {
        int sh = (p->chroma && c > 0) ? 1 : 0;
        if (sh && ((p->Ws & 1) || (p->Ht & 1))) return ORC_E_PARAM;
        g->shift[c] = sh;
        g->W[c] = p->Ws >> sh;
        g->H[c] = p->Ht >> sh;
        if (g->W[c] < 1 || g->H[c] < 1 || (g->W[c] % p->block) || (g->H[c] % p->block)) return ORC_E_PARAM; /* R23: B must divide the plane size */
        g->nbx[c] = g->W[c] / p->block;
        g->nby[c] = g->H[c] / p->block;
        g->nblk[c] = g->nbx[c] * g->nby[c];
    }
    return ORC_OK;
}

void orc_tree_free(orc_tree *t)
{
    if (!t) return;
    for (int c = 0; c < 3; ++c) {
        for (int L = 0; L <= t->h; ++L) {
            int np = t->UL[L] * t->VL[L];
            if (t->X[c][L]) {
                for (int i = 0; i < np; ++i) free(t->X[c][L][i]);
                free(t->X[c][L]);
            }
            if (L < t->h) {
                if (t->srv[c][L]) {
                    for (int i = 0; i < np; ++i) free(t->srv[c][L][i]);
                    free(t->srv[c][L]);
                }
                free(t->blk[c][L]);
            }
        }
    }
    free(t);
}

void orc_free(void *p) { free(p); }

/* ---------------------------------------------------------------- phase-shifted search
 * PAPER.md:227-248, Eqs. (1)-(2):
 *   Delta-^{xy} = sum_l |B_P(l) - B_R^{xy}(l)| ,  Delta+^{xy} = sum_l |B_P(l) + B_R^{xy}(l)|
 *   Delta- = min over x,y in [-W,W] ; Delta+ likewise ; Delta = min(Delta-, Delta+).
 * R read as 0 outside the image (R8).  Ties (R9): subtractive before additive, then the
 * smallest dy, then the smallest dx.  Rpad is R with a zero border of W samples.
 * The loops run dy, then the B*B samples, then dx innermost (contiguous in Rpad) -- the same
 * sums as Eqs. (1)-(2), accumulated per (dx,dy).
 */
static void search_block_padded(const int16_t *P, int Ws, const int16_t *Rpad, int rstride, int B, int W,
                                int bx, int by, int32_t out[4])
{
    int nd = 2 * W + 1;
    int32_t sm[129], sp[129]; /* W <= 64 */
    int best_m = 0x7fffffff, best_p = 0x7fffffff;
    int mdx = 0, mdy = 0, pdx = 0, pdy = 0;
    for (int dy = -W; dy <= W; ++dy) {
        for (int d = 0; d < nd; ++d) { sm[d] = 0; sp[d] = 0; }
        for (int j = 0; j < B; ++j) {
            const int16_t *prow = P + (size_t)(by * B + j) * Ws + bx * B;
            const int16_t *rrow = Rpad + (size_t)(by * B + j + dy + W) * rstride + bx * B;
            for (int i = 0; i < B; ++i) {
                int pv = prow[i];
                const int16_t *rr = rrow + i; /* rr[d] = R(x + i + (d - W), y + j + dy) */
                for (int d = 0; d < nd; ++d) {
                    int r = rr[d];
                    sm[d] += iabs(pv - r);
                    sp[d] += iabs(pv + r);
                }
            }
        }
        for (int d = 0; d < nd; ++d) {
            if (sm[d] < best_m) { best_m = sm[d]; mdx = d - W; mdy = dy; }
            if (sp[d] < best_p) { best_p = sp[d]; pdx = d - W; pdy = dy; }
        }
    }
    if (best_m <= best_p) { out[0] = 0; out[1] = mdx; out[2] = mdy; out[3] = best_m; }
    else { out[0] = 1; out[1] = pdx; out[2] = pdy; out[3] = best_p; }
}

/* The same search on the half-pel grid (R28): offsets (dx2, dy2) in [-2W, 2W]^2 half pixels, the reference block interpolated
 * bilinearly (orc_halfpel).  Ties as above, on the half-pel offsets.  The integer-pel candidates are the even offsets, so the
 * minimum is never above the integer-pel minimum. */
static void search_block_halfpel(const int16_t *P, const int16_t *R, int Ws, int Ht, int B, int W, int bx, int by, int32_t out[4])
{
    const orc_plane_src src = {R, Ws, Ht};
    int best_m = 0x7fffffff, best_p = 0x7fffffff;
    int mdx = 0, mdy = 0, pdx = 0, pdy = 0;
    for (int dy = -2 * W; dy <= 2 * W; ++dy)
        for (int dx = -2 * W; dx <= 2 * W; ++dx) {
            int sm = 0, sp = 0;
            for (int j = 0; j < B; ++j)
                for (int i = 0; i < B; ++i) {
                    const int x = bx * B + i, y = by * B + j;
                    const int pv = P[(size_t)y * Ws + x], r = orc_halfpel(orc_plane_at, &src, 2 * x + dx, 2 * y + dy);
                    sm += iabs(pv - r);
                    sp += iabs(pv + r);
                }
            if (sm < best_m) { best_m = sm; mdx = dx; mdy = dy; }
            if (sp < best_p) { best_p = sp; pdx = dx; pdy = dy; }
        }
    if (best_m <= best_p) { out[0] = 0; out[1] = mdx; out[2] = mdy; out[3] = best_m; }
    else { out[0] = 1; out[1] = pdx; out[2] = pdy; out[3] = best_p; }
}

void orc_search_block_halfpel(const int16_t *P, const int16_t *R, int Ws, int Ht, int B, int W, int bx, int by, int32_t out[4])
{
    search_block_halfpel(P, R, Ws, Ht, B, W, bx, by, out);
}

static int16_t *make_padded(const int16_t *R, int Ws, int Ht, int W, int *rstride)
{
    int stride = Ws + 2 * W;
    int16_t *pad = (int16_t *)calloc((size_t)stride * (size_t)(Ht + 2 * W), sizeof(int16_t));
    if (!pad) return NULL;
    for (int y = 0; y < Ht; ++y) memcpy(pad + (size_t)(y + W) * stride + W, R + (size_t)y * Ws, (size_t)Ws * sizeof(int16_t));
    *rstride = stride;
    return pad;
}

void orc_search_block(const int16_t *P, const int16_t *R, int Ws, int Ht, int B, int W, int bx, int by,
                      int32_t out[4])
{
    int rstride = 0;
    int16_t *pad = make_padded(R, Ws, Ht, W, &rstride);
    if (!pad) { out[0] = out[1] = out[2] = 0; out[3] = -1; return; }
    search_block_padded(P, Ws, pad, rstride, B, W, bx, by, out);
    free(pad);
}

static int block_energy(const int16_t *P, int Ws, int B, int bx, int by)
{
    int e = 0;
    for (int j = 0; j < B; ++j)
        for (int i = 0; i < B; ++i) e += iabs(P[(size_t)(by * B + j) * Ws + bx * B + i]);
    return e;
}

/* ---------------------------------------------------------------- encode_begin */
orc_tree *orc_encode_begin(const uint8_t *lf, const orc_params *p, int *err)
{
    int e_dummy;
    if (!err) err = &e_dummy;
    *err = ORC_OK;
    if (!lf || !p || p->U < 1 || p->V < 1 || p->Ws < 1 || p->Ht < 1 || p->height < 1 || p->height > ORC_MAX_LEVELS ||
        p->block < 1 || p->block > 8 || p->window < 0 || p->window > 64 || p->chroma > 1 || p->subpel > 1) {
        *err = ORC_E_PARAM;
        return NULL;
    }
    orc_geom geom;
    if (orc__geom(p, &geom) != ORC_OK) { *err = ORC_E_PARAM; return NULL; }
    orc_tree *t = (orc_tree *)calloc(1, sizeof(orc_tree));
    if (!t) { *err = ORC_E_NOMEM; return NULL; }
    t->p = *p;
    t->g = geom;
    t->h = p->height;
    const int Ws = p->Ws, Ht = p->Ht, B = p->block, W = p->window, h = t->h;
    const size_t npx = (size_t)Ws * Ht;
    for (int L = 0; L <= h; ++L) {
        t->UL[L] = (p->U + (1 << L) - 1) >> L; /* U_L = ceil(U / 2^L)  (R1, R3) */
        t->VL[L] = (p->V + (1 << L) - 1) >> L;
    }
#ifdef _OPENMP
    if (p->nthreads > 0) omp_set_num_threads(p->nthreads);
#endif
    for (int c = 0; c < 3; ++c) {
        const size_t npc = (size_t)t->g.W[c] * t->g.H[c];
        for (int L = 0; L <= h; ++L) {
            int np = t->UL[L] * t->VL[L];
            t->X[c][L] = (int16_t **)calloc((size_t)np, sizeof(int16_t *));
            if (!t->X[c][L]) goto nomem;
            for (int i = 0; i < np; ++i)
                if (!(t->X[c][L][i] = (int16_t *)malloc(npc * sizeof(int16_t)))) goto nomem;
            if (L < h) {
                t->srv[c][L] = (int16_t **)calloc((size_t)np, sizeof(int16_t *));
                if (!t->srv[c][L]) goto nomem;
                for (int i = 0; i < np; ++i)
                    if (!(t->srv[c][L][i] = (int16_t *)malloc(npc * sizeof(int16_t)))) goto nomem;
                t->blk[c][L] = (orc_block *)calloc((size_t)np * t->g.nblk[c], sizeof(orc_block));
                if (!t->blk[c][L]) goto nomem;
            }
        }
    }
    /* step 1: colour, X_0; with p.chroma the Co / Cg planes are reduced by the 2 x 2 box mean (R18) */
    {
        int nviews = p->U * p->V;
        int failed = 0;
#pragma omp parallel for schedule(static)
        for (int vi = 0; vi < nviews; ++vi) {
            const uint8_t *src = lf + (size_t)vi * npx * 3;
            int16_t *full[3] = {t->X[0][0][vi], NULL, NULL};
            if (p->chroma) {
                full[1] = (int16_t *)malloc(npx * sizeof(int16_t));
                full[2] = (int16_t *)malloc(npx * sizeof(int16_t));
                if (!full[1] || !full[2]) { free(full[1]); free(full[2]); failed = 1; continue; }
            } else { full[1] = t->X[1][0][vi]; full[2] = t->X[2][0][vi]; }
            for (size_t i = 0; i < npx; ++i) {
                int y, co, cg;
                orc_rgb_to_ycocg(src[3 * i], src[3 * i + 1], src[3 * i + 2], &y, &co, &cg);
                full[0][i] = (int16_t)y;
                full[1][i] = (int16_t)co;
                full[2][i] = (int16_t)cg;
            }
            if (p->chroma) {
                for (int c = 1; c < 3; ++c) {
                    const int Wc = t->g.W[c], Hc = t->g.H[c];
                    for (int y = 0; y < Hc; ++y)
                        for (int x = 0; x < Wc; ++x) {
                            const int16_t *q = full[c] + (size_t)(2 * y) * Ws + 2 * x;
                            t->X[c][0][vi][(size_t)y * Wc + x] = (int16_t)round_mean(q[0] + q[1] + q[Ws] + q[Ws + 1], 4);
                        }
                    free(full[c]);
                }
            }
        }
        if (failed) goto nomem;
    }
    /* step 2: hierarchy: RKV = filtered cluster, SRV = member - RKV, recurse */
    for (int c = 0; c < 3; ++c) {
        const size_t npc = (size_t)t->g.W[c] * t->g.H[c];
        for (int L = 0; L < h; ++L) {
            int UL = t->UL[L], VL = t->VL[L], UP = t->UL[L + 1], VP = t->VL[L + 1];
#pragma omp parallel for schedule(static)
            for (int q = 0; q < UP * VP; ++q) {
                int qu = q % UP, qv = q / UP;
                const int16_t *mem[4];
                int16_t *srvp[4];
                int n = 0;
                for (int j = 0; j < 2; ++j)
                    for (int i = 0; i < 2; ++i) {
                        int pu = 2 * qu + i, pv = 2 * qv + j;
                        if (pu < UL && pv < VL) { mem[n] = t->X[c][L][pv * UL + pu]; srvp[n] = t->srv[c][L][pv * UL + pu]; ++n; }
                    }
                int16_t *rk = t->X[c][L + 1][q];
                for (size_t i = 0; i < npc; ++i) {
                    int s = 0;
                    for (int k = 0; k < n; ++k) s += mem[k][i];
                    int r = round_mean(s, n);
                    rk[i] = (int16_t)r;
                    for (int k = 0; k < n; ++k) srvp[k][i] = (int16_t)(mem[k][i] - r);
                }
            }
        }
    }
    /* steps 3-4: roles (R5: the even-even member of each cluster is the reference) and the
     * exhaustive phase-shifted search of every block of every predictive plane against the
     * UNTHRESHOLDED reference SRV of its cluster (R12 open loop). */
    for (int c = 0; c < 3; ++c) {
        const int Wc = t->g.W[c], Hc = t->g.H[c], nbx = t->g.nbx[c], nby = t->g.nby[c], nblk = t->g.nblk[c];
        for (int L = 0; L < h; ++L) {
            int UL = t->UL[L], VL = t->VL[L];
            /* block energies for all planes */
#pragma omp parallel for schedule(static)
            for (int pi = 0; pi < UL * VL; ++pi) {
                orc_block *bk = t->blk[c][L] + (size_t)pi * nblk;
                for (int by = 0; by < nby; ++by)
                    for (int bx = 0; bx < nbx; ++bx) bk[by * nbx + bx].E = block_energy(t->srv[c][L][pi], Wc, B, bx, by);
            }
            for (int rv = 0; rv < VL; rv += 2)
                for (int ru = 0; ru < UL; ru += 2) {
                    int rstride = 0;
                    int16_t *pad = make_padded(t->srv[c][L][rv * UL + ru], Wc, Hc, W, &rstride);
                    if (!pad) goto nomem;
                    for (int j = 0; j < 2; ++j)
                        for (int i = 0; i < 2; ++i) {
                            int pu = ru + i, pv = rv + j;
                            if ((i | j) == 0 || pu >= UL || pv >= VL) continue;
                            const int16_t *P = t->srv[c][L][pv * UL + pu];
                            orc_block *bk = t->blk[c][L] + (size_t)(pv * UL + pu) * nblk;
#pragma omp parallel for schedule(dynamic, 4)
                            for (int b = 0; b < nblk; ++b) {
                                int32_t r[4];
                                if (p->subpel) search_block_halfpel(P, t->srv[c][L][rv * UL + ru], Wc, Hc, B, W, b % nbx, b / nbx, r);
                                else search_block_padded(P, Wc, pad, rstride, B, W, b % nbx, b / nbx, r);
                                bk[b].mode = r[0]; bk[b].dx = r[1]; bk[b].dy = r[2]; bk[b].sad = r[3];
                            }
                        }
                    free(pad);
                }
        }
    }
    orc_tree_threshold(t, p->tau_ref, p->tau_res, p->policy);
    return t;
nomem:
    orc_tree_free(t);
    *err = ORC_E_NOMEM;
    return NULL;
}
