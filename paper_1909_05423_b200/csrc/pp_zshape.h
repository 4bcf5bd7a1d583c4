// Host-side size rules of the z solve: which kernel family takes which nz (no device code here, so the plan
// code can include it without pulling in the kernels).
#pragma once

namespace pp {

constexpr int Z_MAX_BATCH = 64;   // grids per launch of the batched one-CTA partitioned kernel (pp_solve_batch)
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
#ifndef PP_Z1024_R
#define PP_Z1024_R 64
#define PP_Z1024_L 16
#endif
    if (nz == 1024) return {PP_Z1024_R, 1024 / PP_Z1024_R, PP_Z1024_L};
    if (nz == 2048) return {64, 32, 8};
    return {0, 0, 0};
}

// long lines: super-segments of 256 rows (R = 32, S = 8), nz a multiple of 256, at least two of them
constexpr int ZP_HIER_ROWS = 256;
inline bool zpart_hier_ok(int nz) { return nz % ZP_HIER_ROWS == 0 && nz / ZP_HIER_ROWS >= 2 && nz <= 16384; }

// ... and, Neumann / Dirichlet z with at most 8 super-segments (the portable thread-block cluster size), both levels in one
// pass by a cluster of nz / 256 CTAs per line (zsolve_part_kernel MODE 3).  Measured (256 x 256 planes, GB/s over 16 B per
// point): nz = 768: 3516 against 3293 for the two-level passes; 1280: 3451 / 3391; 2048: 3298 against 2999 for one CTA
// per line; but 1024: 3537 against 4052 for one CTA per line (64 rows per thread), and 2706 / 3040 on a 128 x 128 plane
// (too few clusters) -- hence the rule below.
#ifndef PP_Z_CLUSTER_MIN
#define PP_Z_CLUSTER_MIN 768         // shortest line that takes the cluster kernel
#endif
#ifndef PP_Z_CLUSTER_MIN_PLANE
#define PP_Z_CLUSTER_MIN_PLANE 32768 // fewest lines
#endif
inline bool zpart_cluster_possible(int nz, bool periodic) {
    return !periodic && nz % ZP_HIER_ROWS == 0 && nz / ZP_HIER_ROWS >= 2 && nz / ZP_HIER_ROWS <= 8;
}
inline bool zpart_cluster_ok(int nz, long long plane, bool periodic) {
    return zpart_cluster_possible(nz, periodic) && nz >= PP_Z_CLUSTER_MIN && nz != 1024 && plane >= PP_Z_CLUSTER_MIN_PLANE;
}

}  // namespace pp
