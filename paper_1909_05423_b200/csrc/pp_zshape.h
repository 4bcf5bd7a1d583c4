// Host-side size rules of the z solve: which kernel family takes which nz (no device code here, so the plan
// code can include it without pulling in the kernels).
#pragma once

namespace pp {

constexpr int Z_MAX_CK = 64;   // checkpoints per line of the two-sweep kernels (nz <= 64 Z_MAX_CK)

struct ZPartShape {
    int R, S, L;              // rows per thread, segments per system, systems per CTA
};

// which (R, S, L) serves this nz; R == 0: not supported by the partitioned kernel
#ifndef PP_ZP_MAXT
#define PP_ZP_MAXT 256    // threads per CTA (L S) never exceeds this
#define PP_ZP_MINB 2      // resident CTAs per SM the R = 32 kernel is compiled for (R = 64: half)
#endif
#ifndef PP_ZP_L
#define PP_ZP_L 32        // systems per CTA when S <= 8
#endif
inline ZPartShape zpart_shape(int nz) {
    if (nz % 32 == 0 && nz / 32 <= 8) return {32, nz / 32, PP_ZP_L};
    if (nz % 64 == 0 && nz / 64 <= 8) return {64, nz / 64, PP_ZP_L};
    if (nz == 1024) return {64, 16, 16};
    if (nz == 2048) return {64, 32, 8};
    return {0, 0, 0};
}

// long lines: super-segments of 256 rows (R = 32, S = 8), nz a multiple of 256, at least two of them
constexpr int ZP_HIER_ROWS = 256;
inline bool zpart_hier_ok(int nz) { return nz % ZP_HIER_ROWS == 0 && nz / ZP_HIER_ROWS >= 2 && nz <= 16384; }

}  // namespace pp
