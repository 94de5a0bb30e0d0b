/* Brute-force density of states of the 4x4 periodic 3-state Potts lattice (3^16 states).
 * Test helper (pin of reading D26): independent of oracle/ and of the CUDA path.
 * g[B][N0] = number of states with B = number of nearest-neighbour bonds joining equal states (each of the
 * 32 bonds once) and N0 = number of sites in state 0.                                                      */
#include <stdint.h>
#include <string.h>
void enum_potts3_4x4(int64_t *g /* [33][17] */)
{
    int s[16];
    memset(g, 0, sizeof(int64_t) * 33 * 17);
    for (long code = 0; code < 43046721L; ++code) {
        long c = code;
        for (int i = 0; i < 16; ++i) { s[i] = (int)(c % 3); c /= 3; }
        int B = 0, N0 = 0;
        for (int y = 0; y < 4; ++y)
            for (int x = 0; x < 4; ++x) {
                int v = s[x + 4 * y];
                B += (v == s[(x + 1) % 4 + 4 * y]) + (v == s[x + 4 * ((y + 1) % 4)]);
                N0 += (v == 0);
            }
        g[B * 17 + N0] += 1;
    }
}
