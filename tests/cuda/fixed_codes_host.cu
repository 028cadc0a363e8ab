// Host-only check of the dictionary lattice's fixed codes (rms_internal.cuh: rms_fixed_code / rms_fixed_word), compiled and run by
// tests/test_host_side.py (no GPU needed).  Prints one line: the number of violations found and a few counts.
#include <cstdio>
#include "../../paper_2012_06478_b200/csrc/rms_internal.cuh"

static bool invariant_along(uint32_t m, int axis)
{
    // the same-label bit of (dx, dy, dz) does not depend on the coordinate along `axis` (0 = x, 1 = y, 2 = z)
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            int bits[3];
            for (int t = 0; t < 3; ++t) {
                const int dx = axis == 0 ? t : a, dy = axis == 1 ? t : (axis == 0 ? a : b), dz = axis == 2 ? t : b;
                bits[t] = (m >> (dx + 3 * dy + 9 * dz)) & 1u;
            }
            if (bits[0] != bits[1] || bits[1] != bits[2]) return false;
        }
    return true;
}

int main()
{
    int bad = 0, n_fixed = 0;
    // every fixed code: its word maps back to it (or, where a word is invariant along two axes, to the first family that
    // matches, whose word is the same), carries the centre bit, and is invariant along the family's axis
    for (uint32_t code = 0; code < RMS_DICT_FIXED; ++code) {
        const uint32_t w = rms_fixed_word(code);
        if (!w) continue;
        ++n_fixed;
        const uint32_t c = rms_fixed_code(w);
        if (c == RMS_DICT_NONE || rms_fixed_word(c) != w) ++bad;
        if (!((w >> RMS_NBR_SELF) & 1u)) ++bad;
        if (((w & RMS_NBR_GHOST) != 0u) != (code >= 1024u)) ++bad;
        const uint32_t k = code & 1023u;
        if (k >= 1u && k <= 768u && !invariant_along(w & 0x07FFFFFFu, 2 - (int)((k - 1u) >> 8))) ++bad;
    }
    if (rms_fixed_code(0x07FFFFFFu) != 0u || rms_fixed_code(0x07FFFFFFu | RMS_NBR_GHOST) != 1024u) ++bad;
    // pseudo-random words: a code only where the word really is invariant along an axis, and then the right word back
    uint32_t x = 12345u;
    int hits = 0;
    for (int i = 0; i < 4000000; ++i) {
        x = x * 1664525u + 1013904223u;
        uint32_t m = ((x >> 4) & 0x07FFFFFFu) | (1u << RMS_NBR_SELF);
        if ((i & 3) == 0) m &= ~(x & 0x00492492u) | (1u << RMS_NBR_SELF);       // some sparser words
        const uint32_t c = rms_fixed_code(m);
        const bool inv = invariant_along(m, 0) || invariant_along(m, 1) || invariant_along(m, 2);
        if ((c != RMS_DICT_NONE) != inv) ++bad;
        if (c != RMS_DICT_NONE) { ++hits; if (rms_fixed_word(c) != m) ++bad; }
    }
    // every word that is invariant along z: built from each 3 x 3 cross-section
    for (uint32_t q = 0; q < 512u; ++q) {
        if (!((q >> 4) & 1u)) continue;
        const uint32_t m = q | (q << 9) | (q << 18);
        const uint32_t c = rms_fixed_code(m);
        if (c == RMS_DICT_NONE || rms_fixed_word(c) != m) ++bad;
    }
    printf("bad %d fixed %d hits %d\n", bad, n_fixed, hits);
    return bad != 0;
}
