// tm_gamma.cuh -- the library's own gamma tables (chiral basis of include/tm.h), multiplied out in integer arithmetic on the
// host.  Gamma_n = g1^b0 g2^b1 g3^b2 g4^b3, n = b0 + 2 b1 + 4 b2 + 8 b3 (reading 15).
#pragma once

namespace tmk {

struct GammaZ { int re, im; };

// g[mu][al][be], mu = 0..3 = x,y,z,t: g_k = [[0, -i s_k], [i s_k, 0]], g_4 = [[0, 1], [1, 0]]
static inline void gamma_mu_table(GammaZ g[4][4][4])
{
    auto mul = [](GammaZ a, GammaZ b) { return GammaZ{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; };
    for (int m = 0; m < 4; ++m)
        for (int a = 0; a < 4; ++a)
            for (int b = 0; b < 4; ++b) g[m][a][b] = GammaZ{0, 0};
    const GammaZ s[3][2][2] = {{{{0, 0}, {1, 0}}, {{1, 0}, {0, 0}}}, {{{0, 0}, {0, -1}}, {{0, 1}, {0, 0}}}, {{{1, 0}, {0, 0}}, {{0, 0}, {-1, 0}}}};
    for (int k = 0; k < 3; ++k)
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b) {
                g[k][a][2 + b] = mul(GammaZ{0, -1}, s[k][a][b]);
                g[k][2 + a][b] = mul(GammaZ{0, 1}, s[k][a][b]);
            }
    g[3][0][2] = g[3][1][3] = g[3][2][0] = g[3][3][1] = GammaZ{1, 0};
}

struct GammaTable {
    // Gamma_n has one non-zero entry per row: (Gamma_n)_{al, col[n][al]} = re + i im, entries in {+-1, +-i}
    signed char col[16][4], re[16][4], im[16][4];
};

static inline GammaTable make_gamma_table()
{
    auto mul = [](GammaZ a, GammaZ b) { return GammaZ{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; };
    GammaZ g[4][4][4];
    gamma_mu_table(g);
    GammaTable tb;
    for (int n = 0; n < 16; ++n) {
        GammaZ p[4][4] = {};
        for (int a = 0; a < 4; ++a) p[a][a] = GammaZ{1, 0};
        for (int k = 0; k < 4; ++k) {
            if (!((n >> k) & 1)) continue;
            GammaZ q[4][4] = {};
            for (int a = 0; a < 4; ++a)
                for (int b = 0; b < 4; ++b)
                    for (int c = 0; c < 4; ++c) {
                        const GammaZ m = mul(p[a][c], g[k][c][b]);
                        q[a][b].re += m.re;
                        q[a][b].im += m.im;
                    }
            for (int a = 0; a < 4; ++a)
                for (int b = 0; b < 4; ++b) p[a][b] = q[a][b];
        }
        for (int a = 0; a < 4; ++a)
            for (int b = 0; b < 4; ++b)
                if (p[a][b].re != 0 || p[a][b].im != 0) {
                    tb.col[n][a] = (signed char)b;
                    tb.re[n][a] = (signed char)p[a][b].re;
                    tb.im[n][a] = (signed char)p[a][b].im;
                }
    }
    return tb;
}

} // namespace tmk
