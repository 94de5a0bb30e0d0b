/* Brute-force density of states of the 4x4 periodic spin-1 Ising lattice (3^16 states).
 * Test helper (SURVEY.md 8(c) pin P8): independent of oracle/ and of the CUDA path.
 * g[B+32][M+16][Q] = number of states with bond sum B = sum_<ij> s_i s_j (each bond once,
 * 32 bonds), magnetisation M = sum s_i and Q = sum s_i^2.                                  */
#include <stdint.h>
#include <string.h>
void enum_spin1_4x4(int64_t *g /* [65][33][17] */)
{
    int s[16];
    memset(g, 0, sizeof(int64_t) * 65 * 33 * 17);
    for (long code = 0; code < 43046721L; ++code) {
        long c = code;
        for (int i = 0; i < 16; ++i) { s[i] = (int)(c % 3) - 1; c /= 3; }
        int B = 0, M = 0, Q = 0;
        for (int y = 0; y < 4; ++y)
            for (int x = 0; x < 4; ++x) {
                int v = s[x + 4 * y];
                B += v * (s[(x + 1) % 4 + 4 * y] + s[x + 4 * ((y + 1) % 4)]);
                M += v; Q += v * v;
            }
        g[((B + 32) * 33 + (M + 16)) * 17 + Q] += 1;
    }
}
