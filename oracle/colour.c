/* HMLFC oracle (test infrastructure) -- colour transform.
 *
 * PAPER.md:263 (section 4.5): "YCoCg colour space is used ... The dynamic range (number of
 * bits to store pixels) of the pixel values is adjusted accordingly to avoid any loss of
 * information due to transformations."  Reading R17: the lossless lifting form
 * YCoCg-R with arithmetic (floor) shifts.  Ranges: y in [0,255], co,cg in [-255,255].
 */
#include "hmlfc_oracle.h"

/* floor(x / 2) for signed x, written out so it does not depend on >> of negatives */
static int floor_half(int x) { return (x >= 0) ? (x / 2) : -((-x + 1) / 2); }

void orc_rgb_to_ycocg(int r, int g, int b, int *y, int *co, int *cg)
{
    int Co = r - b;
    int t = b + floor_half(Co);
    int Cg = g - t;
    int Y = t + floor_half(Cg);
    *y = Y;
    *co = Co;
    *cg = Cg;
}

void orc_ycocg_to_rgb(int y, int co, int cg, int *r, int *g, int *b)
{
    int t = y - floor_half(cg);
    int G = cg + t;
    int B = t - floor_half(co);
    int R = B + co;
    *r = R;
    *g = G;
    *b = B;
}

int64_t orc_colour_roundtrip_failures(void)
{
    int64_t bad = 0;
    for (int r = 0; r < 256; ++r)
        for (int g = 0; g < 256; ++g)
            for (int b = 0; b < 256; ++b) {
                int y, co, cg, r2, g2, b2;
                orc_rgb_to_ycocg(r, g, b, &y, &co, &cg);
                orc_ycocg_to_rgb(y, co, cg, &r2, &g2, &b2);
                if (r2 != r || g2 != g || b2 != b) ++bad;
                if (y < 0 || y > 255 || co < -255 || co > 255 || cg < -255 || cg > 255) ++bad;
            }
    return bad;
}
