/* HMLFC oracle (test infrastructure) -- thresholds, stored values (replacement
 * step), the encoder's own dense reconstruction P1 and
 * introspection for the pins. */
#include "oracle_internal.h"

#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------- two-threshold decision
 * "an energy value is computed by summing up the absolute values of the pixels
 * in the block.  If the energy is less than the user set threshold the block is marked as
 * insignificant and not stored"; two independent thresholds for reference and residual SRVs.
 * R11: significant iff energy >= tau.  R13: per predictive block two flags (pred,res).
 */
int orc_tree_threshold(orc_tree *t, int tau_ref, int tau_res, int policy)
{
    if (!t || tau_ref < 0 || tau_res < 0 || policy < 0 || policy > 3) return ORC_E_PARAM;
    t->p.tau_ref = tau_ref;
    t->p.tau_res = tau_res;
    t->p.policy = policy;
    for (int c = 0; c < 3; ++c)
        for (int L = 0; L < t->h; ++L) {
            int UL = t->UL[L], VL = t->VL[L];
            for (int pv = 0; pv < VL; ++pv)
                for (int pu = 0; pu < UL; ++pu) {
                    orc_block *bk = t->blk[c][L] + (size_t)(pv * UL + pu) * t->g.nblk[c];
                    for (int b = 0; b < t->g.nblk[c]; ++b) {
                        int res, pred = 0;
                        if (!orc_is_predictive(pu, pv)) {
                            res = bk[b].E >= tau_ref;
                        } else if (policy == ORC_POLICY_ADAPTIVE) {
                            int worth = bk[b].E >= tau_res;
                            pred = worth && (bk[b].sad < bk[b].E);
                            int e_energy = pred ? bk[b].sad : bk[b].E; /* sum|e| */
                            res = worth && (e_energy >= tau_res);
                        } else if (policy == ORC_POLICY_ALL) {
                            pred = 1;
                            res = bk[b].sad >= tau_res;
                        } else if (policy == ORC_POLICY_LITERAL) {
                            res = bk[b].sad >= tau_res;
                            pred = res;
                        } else { /* ORC_POLICY_NOMOTION: the hierarchy alone (RLFC): predictive planes are coded intra */
                            res = bk[b].E >= tau_res;
                        }
                        bk[b].flags = (res ? 1 : 0) | (pred ? 2 : 0);
                    }
                }
        }
    t->thresholded = 1;
    return ORC_OK;
}

/* value of plane (L,pu,pv,c) as STORED in the HMLFC tree at pixel (x,y) of that channel's plane, ignoring the res flag:
 * reference plane: the SRV sample; predictive plane: e = P - (pred ? +-R(x+dx,y+dy) : 0) with the
 * unthresholded reference R (R12), R = 0 outside the image (R8).  R10: sub: e = P - R; add: e = P + R. */
static int stored_value(const orc_tree *t, int c, int L, int pu, int pv, int x, int y)
{
    int UL = t->UL[L];
    int B = t->p.block;
    const int Wc = t->g.W[c], Hc = t->g.H[c];
    int v = t->srv[c][L][pv * UL + pu][(size_t)y * Wc + x];
    if (!orc_is_predictive(pu, pv)) return v;
    const orc_block *bk = t->blk[c][L] + (size_t)(pv * UL + pu) * t->g.nblk[c] + (y / B) * t->g.nbx[c] + (x / B);
    if (bk->flags & 2) {
        const orc_plane_src src = {t->srv[c][L][(pv & ~1) * UL + (pu & ~1)], Wc, Hc};
        const int r = t->p.subpel ? orc_halfpel(orc_plane_at, &src, 2 * x + bk->dx, 2 * y + bk->dy)  /* R28: offsets in half pixels */
                                  : orc_plane_at(&src, x + bk->dx, y + bk->dy);
        v = bk->mode ? v + r : v - r;
    }
    return v;
}

int orc_tree_level_dims(const orc_tree *t, int L, int *UL, int *VL)
{
    if (!t || L < 0 || L > t->h) return ORC_E_PARAM;
    *UL = t->UL[L];
    *VL = t->VL[L];
    return ORC_OK;
}

int orc_tree_get_plane(const orc_tree *t, int kind, int L, int pu, int pv, int c, int16_t *out)
{
    if (!t || c < 0 || c > 2 || L < 0 || L > t->h || (kind != 0 && L >= t->h)) return ORC_E_PARAM;
    if (pu < 0 || pv < 0 || pu >= t->UL[L] || pv >= t->VL[L]) return ORC_E_PARAM;
    size_t npx = (size_t)t->g.W[c] * t->g.H[c];  /* the channel's own plane size (R18) */
    if (kind == 0) memcpy(out, t->X[c][L][pv * t->UL[L] + pu], npx * sizeof(int16_t));
    else if (kind == 1) memcpy(out, t->srv[c][L][pv * t->UL[L] + pu], npx * sizeof(int16_t));
    else if (kind == 2) {
        for (int y = 0; y < t->g.H[c]; ++y)
            for (int x = 0; x < t->g.W[c]; ++x) out[(size_t)y * t->g.W[c] + x] = (int16_t)stored_value(t, c, L, pu, pv, x, y);
    } else return ORC_E_PARAM;
    return ORC_OK;
}

int orc_tree_get_blocks(const orc_tree *t, int L, int pu, int pv, int c, int32_t *out)
{
    if (!t || c < 0 || c > 2 || L < 0 || L >= t->h) return ORC_E_PARAM;
    if (pu < 0 || pv < 0 || pu >= t->UL[L] || pv >= t->VL[L]) return ORC_E_PARAM;
    const orc_block *bk = t->blk[c][L] + (size_t)(pv * t->UL[L] + pu) * t->g.nblk[c];
    for (int b = 0; b < t->g.nblk[c]; ++b) {
        out[6 * b + 0] = bk[b].mode; out[6 * b + 1] = bk[b].dx; out[6 * b + 2] = bk[b].dy;
        out[6 * b + 3] = bk[b].sad;  out[6 * b + 4] = bk[b].E;  out[6 * b + 5] = bk[b].flags;
    }
    return ORC_OK;
}

/* internal accessor used by the serialiser (stream.c) */
int orc__stored_value(const orc_tree *t, int c, int L, int pu, int pv, int x, int y)
{
    return stored_value(t, c, L, pu, pv, x, y);
}

/* ---------------------------------------------------------------- P1 dense reconstruction
 * Y_h = X_h ;  Y_L[p] = Y_{L+1}[parent p] + SRV'_L[p]
 *   reference plane : SRV' = stored blocks (0 where res = 0)
 *   predictive plane: SRV' = e*res + (pred ? +-R'_shifted : 0), R' = the STORED (thresholded) reference
 * then inverse colour and clamp (R19).
 */
int orc_tree_reconstruct(const orc_tree *t, uint8_t *lf_out)
{
    if (!t || !lf_out || !t->thresholded) return ORC_E_PARAM;
    const int B = t->p.block, h = t->h;
    const int nviews = t->p.U * t->p.V;
    int16_t *Y0[3];
    for (int c = 0; c < 3; ++c) Y0[c] = NULL;
    for (int c = 0; c < 3; ++c) {
        /* every channel at its own resolution (R18) */
        const int Ws = t->g.W[c], Ht = t->g.H[c], nbx = t->g.nbx[c], nblk = t->g.nblk[c];
        const size_t npx = (size_t)Ws * Ht;
        /* Y[L] arrays of planes, built top-down */
        int16_t *above = (int16_t *)malloc((size_t)t->UL[h] * t->VL[h] * npx * sizeof(int16_t));
        if (!above) return ORC_E_NOMEM;
        for (int i = 0; i < t->UL[h] * t->VL[h]; ++i) memcpy(above + (size_t)i * npx, t->X[c][h][i], npx * sizeof(int16_t));
        for (int L = h - 1; L >= 0; --L) {
            int UL = t->UL[L], VL = t->VL[L], UP = t->UL[L + 1];
            int16_t *cur = (int16_t *)malloc((size_t)UL * VL * npx * sizeof(int16_t));
            int16_t *Rp = (int16_t *)malloc(npx * sizeof(int16_t)); /* R' of the current cluster */
            if (!cur || !Rp) { free(cur); free(Rp); free(above); return ORC_E_NOMEM; }
            for (int rv = 0; rv < VL; rv += 2)
                for (int ru = 0; ru < UL; ru += 2) {
                    /* stored reference R' */
                    const orc_block *rb = t->blk[c][L] + (size_t)(rv * UL + ru) * nblk;
                    const int16_t *rs = t->srv[c][L][rv * UL + ru];
                    for (int y = 0; y < Ht; ++y)
                        for (int x = 0; x < Ws; ++x)
                            Rp[(size_t)y * Ws + x] = (rb[(y / B) * nbx + (x / B)].flags & 1) ? rs[(size_t)y * Ws + x] : 0;
                    for (int j = 0; j < 2; ++j)
                        for (int i = 0; i < 2; ++i) {
                            int pu = ru + i, pv = rv + j;
                            if (pu >= UL || pv >= VL) continue;
                            const int16_t *par = above + (size_t)((pv >> 1) * UP + (pu >> 1)) * npx;
                            int16_t *dst = cur + (size_t)(pv * UL + pu) * npx;
                            const orc_block *bk = t->blk[c][L] + (size_t)(pv * UL + pu) * nblk;
                            for (int y = 0; y < Ht; ++y)
                                for (int x = 0; x < Ws; ++x) {
                                    int s;
                                    if ((i | j) == 0) s = Rp[(size_t)y * Ws + x];
                                    else {
                                        const orc_block *b = bk + (y / B) * nbx + (x / B);
                                        s = (b->flags & 1) ? stored_value(t, c, L, pu, pv, x, y) : 0;
                                        if (b->flags & 2) {
                                            const orc_plane_src src = {Rp, Ws, Ht};
                                            const int q = t->p.subpel ? orc_halfpel(orc_plane_at, &src, 2 * x + b->dx, 2 * y + b->dy)
                                                                      : orc_plane_at(&src, x + b->dx, y + b->dy);
                                            s += b->mode ? -q : q;
                                        }
                                    }
                                    dst[(size_t)y * Ws + x] = (int16_t)(par[(size_t)y * Ws + x] + s);
                                }
                        }
                }
            free(Rp);
            free(above);
            above = cur;
        }
        Y0[c] = above;
    }
    /* inverse colour at full resolution; a subsampled chroma plane is replicated (nearest neighbour, R18) */
    const int Wf = t->p.Ws, Hf = t->p.Ht;
    for (int vi = 0; vi < nviews; ++vi)
        for (int y = 0; y < Hf; ++y)
          for (int x = 0; x < Wf; ++x) {
            int r, g, b, a[3];
            for (int c = 0; c < 3; ++c)
                a[c] = Y0[c][(size_t)vi * t->g.W[c] * t->g.H[c] + (size_t)(y >> t->g.shift[c]) * t->g.W[c] + (x >> t->g.shift[c])];
            orc_ycocg_to_rgb(a[0], a[1], a[2], &r, &g, &b);
            uint8_t *o = lf_out + (((size_t)vi * Hf + y) * Wf + x) * 3;
            o[0] = (uint8_t)(r < 0 ? 0 : (r > 255 ? 255 : r));
            o[1] = (uint8_t)(g < 0 ? 0 : (g > 255 ? 255 : g));
            o[2] = (uint8_t)(b < 0 ? 0 : (b > 255 ? 255 : b));
        }
    for (int c = 0; c < 3; ++c) free(Y0[c]);
    return ORC_OK;
}
