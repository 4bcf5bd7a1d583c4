// z-solve, register-resident partitioned variant: the same tridiagonal systems as pp_zsolve.cuh
// (Algorithm 2), each read from HBM once and written once.
//
// The Thomas sweep of pp_zsolve.cuh touches every unknown twice (forward x', backward x) and
// relies on the L2 to keep x' between the sweeps.  Here a z line of nz = R S rows is cut into S
// segments of R rows; S threads own one system, each keeps its R right-hand sides in registers,
// and the segments are coupled by the partition ("spike") form of the elimination -- the same
// arithmetic the paper's CR-P reduction phase does across ranks, done across
// the threads of one CTA:
//
//   segment block B (R x R, diagonal d_i, off-diagonals 1), neighbours xl = x_{a-1}, xr = x_{a+R}:
//       x_loc = y - v xl - w xr,      y = B^-1 r_loc,  v = B^-1 e_0,  w = B^-1 e_{R-1}
//   With the leading minors q_0 = 1, q_1 = d_0, q_{i+1} = d_i q_i - q_{i-1} (det B = q_R):
//       Thomas pivots  g_i = q_i / q_{i+1}                      (g_k = 1/beta_k of Algorithm 1)
//       w_i = (-1)^(R-1-i) q_i / q_R,   v_i = (-1)^i q_{R-1-i} / q_R  (Toeplitz block)
//   so one table of q per system serves the pivots and both spikes.  Only two distinct blocks
//   exist per system: the interior block (all d_i = b) and the first block (d_0 = b_end); the last
//   block is the first one mirrored, and its owner simply holds its rows in reverse order.
//
//   The 2(S-1) interface unknowns (last row of segment J, first row of segment J+1) satisfy a
//   block-tridiagonal system with 2x2 blocks.  Its matrix depends on the mode only, so it is
//   factored (the divisions) while the loads are still in flight; the right-hand-side part is a
//   short FMA chain run by one thread per system through shared memory.  Every segment then
//   applies  x_i = y_i - v_i xl - w_i xr  and stores.
//
// Thread mapping: CTA = L lanes x S segments; lane l owns system blockIdx.x L + l (consecutive x:
// every row access of a segment is one coalesced L*8-byte run), thread (l, j) owns rows
// [j R, (j+1) R).  All R loads of a thread are issued before anything else, so a resident CTA has
// its whole tile (L nz doubles) in flight.
//
// Periodic z (template flag CYC): every segment is an interior block and the interface chain closes on
// itself; the two wrap-around couplings are folded in by a 2x2 closure (see the kernel) -- an exact
// cyclic solve in place of the Sherman-Morrison correction of PAPER.md:216.
//
// nz must be R S with R in {32, 64} (zpart_shape); longer Neumann / Dirichlet lines (nz = 256 m) use the
// same kernel on two levels (ZHier, MODE 1 / 2); everything else keeps the two-sweep kernels of
// pp_zsolve.cuh.  The singular (0,0) line is handled by zero_mode_line exactly as there.
#pragma once
#include <cooperative_groups.h>

#include "pp_zshape.h"
#include "pp_zsolve.cuh"

namespace pp {

// dynamic shared memory of one CTA, in doubles:
//   Q [2][R+1][L]   leading minors of the first (0) and interior (1) block
//   G [2][R][L]     pivots g_i
//   YF, YL [S][L]   first / last row of every segment's local solution; overwritten by the
//                   interface solution (XL[j] = x just above segment j, XR[j] = x just below it)
//   F [6][S][L]     factored interface matrix (right-hand-side independent): vL, vF, D, A D, sc, sa
//   PC, PA [S][L]   right-hand-side part of the interface elimination
//   RQ [2][L]       1 / q_R of the two blocks
//   ZC [4][S][L]    periodic z only: the interface chain's responses to its two wrap-around couplings
//   CL [4][L]       periodic z only: b1 times the inverse of the 2x2 closure matrix
//   cluster mode (MODE 3) only, after RQ:  SUP [3][L] couplings a0, a1, b1 of the 256-row super-segment blocks;
//   AB [2][L] a1, b1 of the interior R-row block; EXT [2][L] x just above / below the super-segment; XG [2][8][L] first /
//   last unknown of every isolated super-segment of the line (each CTA of the cluster stores its two into all of them
//   through distributed shared memory); SF [4][7][L] factored chain of super-segments (D, A D, sc, sa)
inline size_t zpart_smem_bytes(const ZPartShape &z, bool periodic = false, bool cluster = false) {
    return sizeof(double) * (size_t)z.L * (2 * (z.R + 1) + 2 * z.R + 10 * z.S + 2 + (periodic ? 4 * z.S + 4 : 0) + (cluster ? 51 : 0));
}

// keeps the compiler from hoisting a whole unrolled loop's shared-memory loads above it (which
// costs more registers than the cap allows and ends in local-memory spills)
__device__ __forceinline__ void zp_sched_fence() { asm volatile("" ::: "memory"); }

// leading minors of one block: q_0 = 1, q_1 = d_0, q_{i+1} = d_i q_i - q_{i-1}; returns q_{R-1}, q_R
// and, if TABLES, stores q_i to q[i L] and the pivots g_i = q_i / q_{i+1} to g[i L]
template <int R, bool TABLES>
__device__ __forceinline__ void zp_minors(double d0, double dint, double dlast, double *q, double *g, int L,
                                          double &qRm1, double &qR) {
    double qm = 1.0, qc = d0;
    if (TABLES) { q[0] = qm; q[L] = qc; g[0] = fast_rcp(qc); }
#pragma unroll
    for (int i = 1; i < R; ++i) {
        const double qn = fma((i == R - 1) ? dlast : dint, qc, -qm);
        qm = qc;
        qc = qn;
        if (TABLES) { q[(i + 1) * L] = qn; g[i * L] = qm * fast_rcp(qn); }
    }
    qRm1 = qm;
    qR = qc;
}

// Long systems (nz beyond what one CTA holds): the same partition one level up.  The line is cut into
// nK super-segments of R S rows, one CTA each (blockIdx.y), every one an R S x R S block of the same
// Toeplitz matrix:
//   MODE 1  solves each super-segment as if isolated (neighbours = 0) and writes only its first and
//           last unknown to HF[K], HL[K]                                  (reads 8 B/point)
//   zsolve_hier_interface_kernel couples the super-segments: the same 2x2-block interface system,
//           one thread per mode, leaving x just above / below every super-segment in HL[K-1], HF[K+1]
//   MODE 2  solves each super-segment again with those neighbour values moved to the right-hand
//           side and stores the solution                                   (8 B read + 8 B write)
// MODE 0 is the whole line in one CTA (nK = 1).
//   MODE 3  the same two levels in ONE pass for nK <= 8: the nK CTAs of a line form a thread-block cluster
//           (cluster dimensions (1, nK, 1)); each keeps its isolated super-segment solution in registers, publishes
//           its first and last unknown in its shared memory, reads the other CTAs' through distributed shared
//           memory, solves the small chain of super-segments redundantly, and adds the neighbours' contribution to
//           the registers by a second run of the in-CTA interface chain: 8 B read + 8 B written per point.
struct ZHier {
    int nK;                  // super-segments per line
    double *HF, *HL;         // [nK][plane]
    int periodic;            // periodic z: no super-segment is an end of the line, the chain of super-segments closes
};

template <int R, int MODE, bool CYC = false>
__global__ void __launch_bounds__(PP_ZP_MAXT, (R == 32) ? PP_ZP_MINB : PP_ZP_MINB / 2)
zsolve_part_kernel(double *w, ZParams p, int S, int L, ZHier h) {
    static_assert(!CYC || MODE == 0, "periodic z: single-level only");
    static_assert(MODE != 3 || R == 32, "cluster mode: super-segments of 8 x 32 rows");
    static_assert(R % 2 == 0, "the spike signs below assume an even segment length");
    extern __shared__ double zsm[];
    double *Q = zsm;                                  // [2][R+1][L]
    double *G = Q + 2 * (R + 1) * L;                  // [2][R][L]
    double *YF = G + 2 * R * L;                       // [S][L], later XL
    double *YL = YF + S * L;                          // [S][L], later XR
    double *F = YL + S * L;                           // [6][S][L]
    double *PC = F + 6 * S * L, *PA = PC + S * L;
    double *RQ = PA + S * L;                          // [2][L]
    double *ZC = RQ + 2 * L;                          // [4][S][L]
    double *CL = ZC + 4 * S * L;                      // [4][L]
    // MODE 3 (never periodic), after RQ: SUP [3][L], AB [2][L], EXT [2][L], XG [16][L], SF [28][L]
#define ZP_SUP (RQ + 2 * L)
#define ZP_AB (RQ + 5 * L)
#define ZP_EXT (RQ + 7 * L)
#define ZP_XG (RQ + 9 * L)
#define ZP_SF (RQ + 25 * L)
    if (MODE == 3) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");   // "I run": waited for before the first remote store
    const int SL = S * L;
    // Periodic z: every segment is an interior block and the interface chain closes on itself
    // (S interfaces instead of S - 1); see the closure below.
    constexpr bool cyc = CYC;
    const int NI = cyc ? S : S - 1;                   // interfaces

    if (MODE == 0) w += (size_t)blockIdx.y * p.batch_stride;       // pp_solve_batch: one grid per blockIdx.y
    const int l = threadIdx.x % L, j = threadIdx.x / L;
    const size_t plane = (size_t)p.nx * p.ny;
    const size_t e = (size_t)blockIdx.x * L + l;
    const bool live = e < plane;
    const bool pin = !live || (p.singular && e == 0);       // pinned line: computed with a placeholder, never stored
    const int K = (MODE == 0) ? 0 : (int)blockIdx.y;         // super-segment of this CTA
    const bool top_end = !cyc && ((MODE == 0) || (K == 0 && !h.periodic));          // the CTA's rows start at the line's first row
    const bool bot_end = !cyc && ((MODE == 0) || (K == h.nK - 1 && !h.periodic));   // ... end at its last row
    const bool mirror = bot_end && (S > 1) && (j == S - 1);   // line's last segment: rows held in reverse order
    const int c = ((j == 0 && top_end) || (j == S - 1 && bot_end)) ? 0 : 1;   // first (and mirrored last) / interior block
    // row i of the segment lives at row0 + i * step (the mirrored segment walks upwards)
    const ptrdiff_t step = mirror ? -(ptrdiff_t)plane : (ptrdiff_t)plane;
    double *row0 = w + (live ? e : 0) + (((size_t)K * S + j) * R + (mirror ? R - 1 : 0)) * plane;

    // the mode's shift first (the tabulating threads start from it), then every right-hand side of
    // the segment, in flight at once
    const int jint = cyc ? 0 : 1;                             // who tabulates the interior block
    const int jfac = cyc ? ((S >= 2) ? 1 : 0) : ((S >= 3) ? 2 : 1);   // who factors the interface matrix
    double s = -1.0;
    const int jsup = (MODE == 3) ? jfac + 1 : jfac;           // MODE 3: thread jfac+1 factors the chain of super-segments
    if (j <= jsup && !pin) s = __ldg(p.sx + (int)(e % p.nx)) + __ldg(p.sy + (int)(e / p.nx));
    double ext0 = 0.0, ext1 = 0.0;                            // x just above the CTA's first row / below its last
    if (MODE == 2 && live) {
        if (j == 0 && !top_end) ext0 = h.HL[(size_t)((K > 0) ? K - 1 : h.nK - 1) * plane + e];
        if (j == S - 1 && !bot_end) ext1 = h.HF[(size_t)((K + 1 < h.nK) ? K + 1 : 0) * plane + e];
    }
    double y[R];
#pragma unroll
    for (int i = 0; i < R; ++i) y[i] = __ldcg(row0 + i * step);

    // While the loads fly: thread 0 of the system tabulates the first block, thread jint the interior
    // block, thread jfac factors the interface matrix.
    if (j <= jfac) {
        const double bint = -2.0 + s;
        const double bend = ((p.bcz == 1) ? -1.0 : -3.0) + s;
        double qa, qb;
        if (j == 0 && !cyc) {
            zp_minors<R, true>(bend, bint, (S == 1) ? bend : bint, Q + l, G + l, L, qa, qb);
            RQ[l] = fast_rcp(qb);
        } else if (j == jint) {
            zp_minors<R, true>(bint, bint, bint, Q + (R + 1) * L + l, G + R * L + l, L, qa, qb);
            RQ[L + l] = fast_rcp(qb);
        }
        if (j == jfac) {
            // interface system, unknowns a_J = last row of segment J, c_J = first row of segment J+1:
            //   a_J + vL_J a_{J-1} + wL_J c_J         = yL_J
            //   c_J + vF_{J+1} a_J + wF_{J+1} c_{J+1} = yF_{J+1}
            // end blocks:      wL = vF = q_{R-1}/q_R =: a0,  no outward coupling
            // interior blocks: wL = vF = q_{R-1}/q_R =: a1,  vL = wF = (-1)^(R-1)/q_R =: b1
            // block Thomas: with A_J = wL_J - vL_J sa_{J-1}, D_J = 1 / (1 - vF_{J+1} A_J),
            //   c_J = pc_J - sc_J c_{J+1},  a_J = pa_J - sa_J c_{J+1},  sc_J = D_J wF_{J+1},  sa_J = -A_J sc_J;
            // A, D, sc, sa are right-hand-side independent and computed here.
            // (both blocks' minors again, interleaved in one loop: two independent FMA chains)
            double em = 1.0, ec = bend, im = 1.0, ic = bint;
#pragma unroll
            for (int i = 1; i < R; ++i) {
                const double en = fma(bint, ec, -em), in = fma(bint, ic, -im);
                em = ec; ec = en;
                im = ic; ic = in;
            }
            const double rqe = fast_rcp(ec), rqi = fast_rcp(ic);
            const bool interior = S >= 3 || MODE != 0 || cyc;                  // is there an interior-type block at all
            const double a1 = interior ? im * rqi : 0.0, b1 = interior ? -rqi : 0.0;
            const double a0 = em * rqe;
            const double atop = top_end ? a0 : a1, abot = bot_end ? a0 : a1;
            if (MODE == 3) { ZP_AB[l] = a1; ZP_AB[L + l] = b1; }
            // A_J obeys the Moebius recurrence A_0 = a0, A_J = a1 + b1^2 A_{J-1} / (1 - a1 A_{J-1}); carried
            // as the ratio N_J / M_J it is two FMAs per step, and the reciprocals leave the dependency chain:
            //   D_J = M_J / (M_J - vF_J N_J),   (A D)_J = N_J / (M_J - vF_J N_J)
            const double k1 = fma(b1, b1, -a1 * a1);
            double N = atop, M = 1.0;
            for (int J = 0; J < NI; ++J) {
                const double vL = (J == 0) ? 0.0 : b1;
                const double vF = (J == NI - 1) ? abot : a1, wF = (J == NI - 1) ? 0.0 : b1;
                const double r = fast_rcp(fma(-vF, N, M));
                const double D = M * r, AD = N * r;
                double *f = F + J * L + l;
                f[0] = vL; f[SL] = vF; f[2 * SL] = D; f[3 * SL] = AD; f[4 * SL] = D * wF; f[5 * SL] = -AD * wF;
                const double Nn = fma(k1, N, a1 * M), Mn = fma(-a1, N, M);
                N = Nn;
                M = Mn;
            }
            if (cyc) {
                // Closure of the periodic chain.  The full interface matrix is the open chain plus the two
                // wrap-around couplings  b1 a_{S-1} in row a_0  and  b1 c_0 in row c_{S-1}:
                //   x = x0 - (b1 a_{S-1}) z1 - (b1 c_0) z2,   z1 = chain^-1 e(row a_0),  z2 = chain^-1 e(row c_{S-1}),
                // and the two wrapped unknowns follow from the 2x2 system  K (a_{S-1}, c_0)^T = (x0a_{S-1}, x0c_0)^T,
                //   K = [1 + b1 z1a_{S-1},  b1 z2a_{S-1};  b1 z1c_0,  1 + b1 z2c_0].
                // z1, z2 depend on the mode only: solved here with the factors just stored.
                double *z1c = ZC + l, *z1a = z1c + SL, *z2c = z1a + SL, *z2a = z2c + SL;
                double pa1 = 0.0;
                for (int J = 0; J < S; ++J) {                   // forward, both unit right-hand sides
                    const double *f = F + J * L + l;
                    const double Ya = fma(-f[0], pa1, (J == 0) ? 1.0 : 0.0);
                    const double t1 = -f[SL] * Ya;
                    pa1 = fma(-f[3 * SL], t1, Ya);
                    z1c[J * L] = f[2 * SL] * t1;
                    z1a[J * L] = pa1;
                    z2c[J * L] = (J == S - 1) ? f[2 * SL] : 0.0;
                    z2a[J * L] = (J == S - 1) ? -f[3 * SL] : 0.0;
                }
                double c1 = 0.0, c2 = 0.0;
                for (int J = S - 1; J >= 0; --J) {              // backward
                    const double *f = F + J * L + l;
                    const double sc = f[4 * SL], sa = f[5 * SL];
                    z1a[J * L] = fma(-sa, c1, z1a[J * L]);
                    c1 = fma(-sc, c1, z1c[J * L]);
                    z1c[J * L] = c1;
                    z2a[J * L] = fma(-sa, c2, z2a[J * L]);
                    c2 = fma(-sc, c2, z2c[J * L]);
                    z2c[J * L] = c2;
                }
                const double k11 = fma(b1, z1a[(S - 1) * L], 1.0), k12 = b1 * z2a[(S - 1) * L];
                const double k21 = b1 * z1c[0], k22 = fma(b1, z2c[0], 1.0);
                const double rdet = b1 / fma(k11, k22, -k12 * k21);
                CL[l] = k22 * rdet; CL[L + l] = -k12 * rdet; CL[2 * L + l] = -k21 * rdet; CL[3 * L + l] = k11 * rdet;
            }
        }
    }
    if (MODE == 3 && j == jfac + 1) {
        // Couplings of the R S-row super-segment blocks, a = q_{n-1} / q_n and b1 = -1 / q_n at n = R S (as in
        // zsolve_hier_interface_kernel), from the R-row block's by doubling: the minors of a Toeplitz block obey
        // q_{2n} = q_n^2 - q_{n-1}^2 and q_{2n-1} = q_{n-1} (2 q_n - b q_{n-1}), i.e. with rho = q_{n-1} / q_n, sig = 1 / q_n:
        //   rho' = rho (2 - b rho) / (1 - rho^2),   sig' = sig^2 / (1 - rho^2)
        // -- log2 S steps instead of R S.  End block (d_0 = b + dl): its minors are q_n + dl q_{n-1}.
        const double bint = -2.0 + s;
        double qm = 1.0, qc = bint;
#pragma unroll
        for (int i = 1; i < R; ++i) {
            const double qn = fma(bint, qc, -qm);
            qm = qc; qc = qn;
        }
        double sig = fast_rcp(qc), rho = qm * sig;
        for (int n = R; n < R * S; n *= 2) {
            const double r = fast_rcp(fma(-rho, rho, 1.0));
            const double t = rho * r;
            rho = t * fma(-bint, rho, 2.0);
            sig = sig * sig * r;                      // underflows to 0 for strongly dominant modes: the coupling is 0 then
        }
        const double dl = (p.bcz == 1) ? 1.0 : -1.0;    // b_end - b
        const double a1 = rho, b1 = -sig;
        const double a0 = fma(rho, fma(dl, bint, 1.0), -dl) * fast_rcp(fma(dl, rho, 1.0));
        ZP_SUP[l] = a0; ZP_SUP[L + l] = a1; ZP_SUP[2 * L + l] = b1;
        // factored chain of super-segments (the right-hand-side independent part of zsolve_hier_interface_kernel)
        const int nK = h.nK;
        const double k1 = fma(b1, b1, -a1 * a1);
        double N = a0, M = 1.0;
        for (int J = 0; J < nK - 1; ++J) {
            const double vF = (J + 1 == nK - 1) ? a0 : a1, wF = (J + 1 == nK - 1) ? 0.0 : b1;
            const double r = fast_rcp(fma(-vF, N, M));
            const double D = M * r, AD = N * r;
            double *f = ZP_SF + J * L + l;
            f[0] = D; f[7 * L] = AD; f[14 * L] = D * wF; f[21 * L] = -AD * wF;
            const double Nn = fma(k1, N, a1 * M), Mn = fma(-a1, N, M);
            const double nrm = fast_rcp(fabs(Mn) > fabs(Nn) ? Mn : Nn);      // only the ratio N / M matters
            N = Nn * nrm;
            M = Mn * nrm;
        }
    }
    __syncthreads();

    // local solve  y = B^-1 (scale r)  in registers: Algorithm 1 with the tabulated pivots, run from
    // both ends of the segment at once (rows k and R-1-k; two independent dependency chains of half
    // the length).  Eliminating upwards from the far end of a block meets a pure Toeplitz diagonal,
    // i.e. the interior block's pivots -- or, with a single segment, the first block's again.
    {
        constexpr int M = R / 2;
        const double *gt = G + c * R * L + l;
        const double *gb = G + ((S == 1 && !cyc) ? 0 : R * L) + l;
        const double scale = p.scale;
        // interior segment: one pivot table serves both ends (one read).  R = 32 only: at 64 rows per thread it measured 2 % slower
        const bool same = (R == 32) && !CYC && (gt == gb);       // (periodic z: 2 % slower with it)
        {
            const double g1 = gt[0], g2 = same ? g1 : gb[0];
            y[0] = fma(y[0], scale, -ext0) * g1;
            y[R - 1] = fma(y[R - 1], scale, -ext1) * g2;
        }
#pragma unroll
        for (int k = 1; k < M; ++k) {
            const double g1 = gt[k * L], g2 = same ? g1 : gb[k * L];
            y[k] = fma(y[k], scale, -y[k - 1]) * g1;
            y[R - 1 - k] = fma(y[R - 1 - k], scale, -y[R - k]) * g2;
            if (k % 4 == 3) zp_sched_fence();
        }
        // couple the halves:  x_{M-1} + gt x_M = y_{M-1},   x_M + gb x_{M-1} = y_M
        const double gtm = gt[(M - 1) * L], gbm = same ? gtm : gb[(M - 1) * L];
        const double rden = fast_rcp(fma(-gtm, gbm, 1.0));
        const double xa = fma(-gtm, y[M], y[M - 1]) * rden, xb = fma(-gbm, y[M - 1], y[M]) * rden;
        y[M - 1] = xa;
        y[M] = xb;
#pragma unroll
        for (int k = M - 2; k >= 0; --k) {
            const double g1 = gt[k * L], g2 = same ? g1 : gb[k * L];
            y[k] = fma(-g1, y[k + 1], y[k]);
            y[R - 1 - k] = fma(-g2, y[R - 2 - k], y[R - 1 - k]);
            if (k % 4 == 0) zp_sched_fence();
        }
    }

    if (S > 1 || cyc) {
        YF[j * L + l] = mirror ? y[R - 1] : y[0];
        YL[j * L + l] = mirror ? y[0] : y[R - 1];
        __syncthreads();
        if (j == 0) {                                   // right-hand-side part of the interface elimination
            // interface J couples the last row of segment J with the first row of segment JF(J) = J + 1
            // (periodic: modulo S).  The next step's coefficients are fetched before the current step's FMA chain.
            const double *f = F + l;
            double vL = f[0], vF = f[SL], D = f[2 * SL], A = f[3 * SL], yl = YL[l], yf = YF[((S > 1) ? L : 0) + l];
            double pa = 0.0;
            for (int J = 0; J < NI; ++J) {
                const int Jn = (J + 1 < NI) ? J + 1 : J;
                const int JFn = (Jn + 1 < S) ? Jn + 1 : 0;
                const double *fn = F + Jn * L + l;
                const double nvL = fn[0], nvF = fn[SL], nD = fn[2 * SL], nA = fn[3 * SL];
                const double nyl = YL[Jn * L + l], nyf = YF[JFn * L + l];
                const double Ya = fma(-vL, pa, yl);
                const double t = fma(-vF, Ya, yf);
                const double pc = D * t;
                pa = fma(-A, t, Ya);                 // A holds (A D)_J
                PC[J * L + l] = pc;
                PA[J * L + l] = pa;
                vL = nvL; vF = nvF; D = nD; A = nA; yl = nyl; yf = nyf;
            }
            f = F + (NI - 1) * L + l;
            double sc = f[4 * SL], sa = f[5 * SL], pc = PC[(NI - 1) * L + l], pav = PA[(NI - 1) * L + l];
            double cn = 0.0;
            if (!cyc) {
                for (int J = NI - 1; J >= 0; --J) {
                    const int Jn = (J > 0) ? J - 1 : 0;
                    const double *fn = F + Jn * L + l;
                    const double nsc = fn[4 * SL], nsa = fn[5 * SL], npc = PC[Jn * L + l], npa = PA[Jn * L + l];
                    const double cv = fma(-sc, cn, pc);
                    const double av = fma(-sa, cn, pav);
                    YL[J * L + l] = cv;                  // XR of segment J   = first row of segment J+1
                    YF[(J + 1) * L + l] = av;            // XL of segment J+1 = last row of segment J
                    cn = cv;
                    sc = nsc; sa = nsa; pc = npc; pav = npa;
                }
            } else {
                // open-chain solution first (kept in PC, PA), then the closure: x = x0 - (b1 a_{S-1}) z1 - (b1 c_0) z2
                for (int J = NI - 1; J >= 0; --J) {
                    const int Jn = (J > 0) ? J - 1 : 0;
                    const double *fn = F + Jn * L + l;
                    const double nsc = fn[4 * SL], nsa = fn[5 * SL], npc = PC[Jn * L + l], npa = PA[Jn * L + l];
                    const double cv = fma(-sc, cn, pc);
                    PA[J * L + l] = fma(-sa, cn, pav);
                    PC[J * L + l] = cv;
                    cn = cv;
                    sc = nsc; sa = nsa; pc = npc; pav = npa;
                }
                const double x0a = PA[(S - 1) * L + l], x0c = PC[l];
                const double ba = fma(CL[l], x0a, CL[L + l] * x0c), bg = fma(CL[2 * L + l], x0a, CL[3 * L + l] * x0c);
                const double *z1c = ZC + l, *z1a = z1c + SL, *z2c = z1a + SL, *z2a = z2c + SL;
                for (int J = 0; J < S; ++J) {
                    const int JF = (J + 1 < S) ? J + 1 : 0;
                    YL[J * L + l] = fma(-ba, z1c[J * L], fma(-bg, z2c[J * L], PC[J * L + l]));    // XR of segment J
                    YF[JF * L + l] = fma(-ba, z1a[J * L], fma(-bg, z2a[J * L], PA[J * L + l]));   // XL of segment JF
                }
            }
        }
        __syncthreads();
        const double *qc = Q + c * (R + 1) * L + l;
        const double xlg = (j >= 1 || cyc) ? YF[j * L + l] : 0.0;
        const double xrg = (j <= S - 2 || cyc) ? YL[j * L + l] : 0.0;
        const double rq = RQ[c * L + l];
        const double XL = (c == 0) ? 0.0 : xlg * rq;
        const double XR = ((c == 0 && mirror) ? xlg : xrg) * rq;
        // x_i = y_i - v_i xl - w_i xr = y_i - (-1)^i (q_{R-1-i} XL - q_i XR)
        // (rows i and R-1-i need the same two minors: with 32 rows per thread each pair is read once; with 64 rows, and with
        // periodic z, that measured 2 % slower than reading row by row)
        if constexpr (R == 32 && !CYC) {
#pragma unroll
            for (int i = 0; i < R / 2; i += 2) {
                const double a0 = qc[i * L], b0 = qc[(R - 1 - i) * L], a1 = qc[(i + 1) * L], b1 = qc[(R - 2 - i) * L];
                y[i] = fma(a0, XR, fma(-b0, XL, y[i]));
                y[R - 1 - i] = fma(-b0, XR, fma(a0, XL, y[R - 1 - i]));
                y[i + 1] = fma(-a1, XR, fma(b1, XL, y[i + 1]));
                y[R - 2 - i] = fma(b1, XR, fma(-a1, XL, y[R - 2 - i]));
                if (i % 4 == 2) zp_sched_fence();
            }
        } else {
#pragma unroll
            for (int i = 0; i < R; i += 2) {
                y[i] = fma(qc[i * L], XR, fma(-qc[(R - 1 - i) * L], XL, y[i]));
                y[i + 1] = fma(-qc[(i + 1) * L], XR, fma(qc[(R - 2 - i) * L], XL, y[i + 1]));
                if (i % 8 == 6) zp_sched_fence();
            }
        }
    }
    if (MODE == 3) {
        // the right-hand-side part of the interface elimination, run by one thread per system (j == 0): reads YF / YL =
        // first / last row of every segment's local solution, leaves XL / XR (x just above / below each segment) there
        const auto chain = [&]() {
                // interface J couples the last row of segment J with the first row of segment JF(J) = J + 1
                // (periodic: modulo S).  The next step's coefficients are fetched before the current step's FMA chain.
                const double *f = F + l;
                double vL = f[0], vF = f[SL], D = f[2 * SL], A = f[3 * SL], yl = YL[l], yf = YF[((S > 1) ? L : 0) + l];
                double pa = 0.0;
                for (int J = 0; J < NI; ++J) {
                    const int Jn = (J + 1 < NI) ? J + 1 : J;
                    const int JFn = (Jn + 1 < S) ? Jn + 1 : 0;
                    const double *fn = F + Jn * L + l;
                    const double nvL = fn[0], nvF = fn[SL], nD = fn[2 * SL], nA = fn[3 * SL];
                    const double nyl = YL[Jn * L + l], nyf = YF[JFn * L + l];
                    const double Ya = fma(-vL, pa, yl);
                    const double t = fma(-vF, Ya, yf);
                    const double pc = D * t;
                    pa = fma(-A, t, Ya);                 // A holds (A D)_J
                    PC[J * L + l] = pc;
                    PA[J * L + l] = pa;
                    vL = nvL; vF = nvF; D = nD; A = nA; yl = nyl; yf = nyf;
                }
                f = F + (NI - 1) * L + l;
                double sc = f[4 * SL], sa = f[5 * SL], pc = PC[(NI - 1) * L + l], pav = PA[(NI - 1) * L + l];
                double cn = 0.0;
                if (!cyc) {
                    for (int J = NI - 1; J >= 0; --J) {
                        const int Jn = (J > 0) ? J - 1 : 0;
                        const double *fn = F + Jn * L + l;
                        const double nsc = fn[4 * SL], nsa = fn[5 * SL], npc = PC[Jn * L + l], npa = PA[Jn * L + l];
                        const double cv = fma(-sc, cn, pc);
                        const double av = fma(-sa, cn, pav);
                        YL[J * L + l] = cv;                  // XR of segment J   = first row of segment J+1
                        YF[(J + 1) * L + l] = av;            // XL of segment J+1 = last row of segment J
                        cn = cv;
                        sc = nsc; sa = nsa; pc = npc; pav = npa;
                    }
                } else {
                    // open-chain solution first (kept in PC, PA), then the closure: x = x0 - (b1 a_{S-1}) z1 - (b1 c_0) z2
                    for (int J = NI - 1; J >= 0; --J) {
                        const int Jn = (J > 0) ? J - 1 : 0;
                        const double *fn = F + Jn * L + l;
                        const double nsc = fn[4 * SL], nsa = fn[5 * SL], npc = PC[Jn * L + l], npa = PA[Jn * L + l];
                        const double cv = fma(-sc, cn, pc);
                        PA[J * L + l] = fma(-sa, cn, pav);
                        PC[J * L + l] = cv;
                        cn = cv;
                        sc = nsc; sa = nsa; pc = npc; pav = npa;
                    }
                    const double x0a = PA[(S - 1) * L + l], x0c = PC[l];
                    const double ba = fma(CL[l], x0a, CL[L + l] * x0c), bg = fma(CL[2 * L + l], x0a, CL[3 * L + l] * x0c);
                    const double *z1c = ZC + l, *z1a = z1c + SL, *z2c = z1a + SL, *z2a = z2c + SL;
                    for (int J = 0; J < S; ++J) {
                        const int JF = (J + 1 < S) ? J + 1 : 0;
                        YL[J * L + l] = fma(-ba, z1c[J * L], fma(-bg, z2c[J * L], PC[J * L + l]));    // XR of segment J
                        YF[JF * L + l] = fma(-ba, z1a[J * L], fma(-bg, z2a[J * L], PA[J * L + l]));   // XL of segment JF
                    }
                }
        };
        // x_i = y_i - v_i xl - w_i xr with the neighbour values in YF / YL; `outer`: segment 0 / S-1 also have a neighbour
        // outside the CTA (MODE 3: the adjacent super-segments of the cluster)
        const auto apply = [&](bool outer) {
            const double *qc = Q + c * (R + 1) * L + l;
            const double xlg = (j >= 1 || cyc || outer) ? YF[j * L + l] : 0.0;
            const double xrg = (j <= S - 2 || cyc || outer) ? YL[j * L + l] : 0.0;
            const double rq = RQ[c * L + l];
            const double XL = (c == 0) ? 0.0 : xlg * rq;
            const double XR = ((c == 0 && mirror) ? xlg : xrg) * rq;
            // x_i = y_i - v_i xl - w_i xr = y_i - (-1)^i (q_{R-1-i} XL - q_i XR)
    #pragma unroll
            for (int i = 0; i < R / 2; i += 2) {
                const double a0 = qc[i * L], b0 = qc[(R - 1 - i) * L], a1 = qc[(i + 1) * L], b1 = qc[(R - 2 - i) * L];
                y[i] = fma(a0, XR, fma(-b0, XL, y[i]));
                y[R - 1 - i] = fma(-b0, XR, fma(a0, XL, y[R - 1 - i]));
                y[i + 1] = fma(-a1, XR, fma(b1, XL, y[i + 1]));
                y[R - 2 - i] = fma(b1, XR, fma(-a1, XL, y[R - 2 - i]));
                if (i % 4 == 2) zp_sched_fence();
            }
        };
        // y is the solution of the isolated super-segment.  Store its first and last unknown into the shared memory of
        // every CTA of the cluster (distributed shared memory), then solve the chain of super-segments -- the interface
        // system of zsolve_hier_interface_kernel, at most 7 steps, factored above -- redundantly in every CTA.
        namespace cg = cooperative_groups;
        cg::cluster_group cluster = cg::this_cluster();
        const int nK = h.nK;
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");        // every CTA of the cluster runs
        if (j == 0 || j == S - 1) {
            const double first = y[0], last = mirror ? y[0] : y[R - 1];
            for (int q = 0; q < nK; ++q) {
                double *dst = cluster.map_shared_rank(ZP_XG, q);
                if (j == 0) dst[K * L + l] = first;
                if (j == S - 1) dst[(8 + K) * L + l] = last;
            }
        }
        asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
        // (no remote access after this point: a CTA may leave as soon as it is done)
        if (j == 0) {
            constexpr int MAXK = 8;
            const double a0 = ZP_SUP[l], a1 = ZP_SUP[L + l], b1 = ZP_SUP[2 * L + l];
            double pa = 0.0;
            double pc[MAXK], pv[MAXK];
#pragma unroll
            for (int J = 0; J < MAXK - 1; ++J) {
                if (J < nK - 1) {
                    const double vL = (J == 0) ? 0.0 : b1;
                    const double vF = (J + 1 == nK - 1) ? a0 : a1;
                    const double *f = ZP_SF + J * L + l;
                    const double Ya = fma(-vL, pa, ZP_XG[(8 + J) * L + l]);
                    const double t = fma(-vF, Ya, ZP_XG[(J + 1) * L + l]);
                    pa = fma(-f[7 * L], t, Ya);
                    pc[J] = f[0] * t; pv[J] = pa;
                }
            }
            double cn = 0.0, ext0 = 0.0, ext1 = 0.0;
#pragma unroll
            for (int J = MAXK - 2; J >= 0; --J) {
                if (J < nK - 1) {
                    const double *f = ZP_SF + J * L + l;
                    const double cv = fma(-f[14 * L], cn, pc[J]);      // first row of super-segment J + 1
                    const double av = fma(-f[21 * L], cn, pv[J]);      // last row of super-segment J
                    cn = cv;
                    if (J == K) ext1 = cv;
                    if (J == K - 1) ext0 = av;
                }
            }
            // The neighbours' values go to the right-hand side: d r = -ext0 e_first - ext1 e_last, whose local solves are
            // -ext0 v in segment 0 and -ext1 w in segment S-1 (v_0 = w_{R-1} = a1, v_{R-1} = w_0 = b1 of the interior
            // block; an end of the line has ext = 0).  The in-CTA chain then gives the change of every interface value.
            const double ia = ZP_AB[l], ib = ZP_AB[L + l];
            for (int q = 0; q < S; ++q) { YF[q * L + l] = 0.0; YL[q * L + l] = 0.0; }
            YF[l] = -ext0 * ia;
            YL[l] = -ext0 * ib;
            YF[(S - 1) * L + l] += -ext1 * ib;
            YL[(S - 1) * L + l] += -ext1 * ia;
            ZP_EXT[l] = ext0;
            ZP_EXT[L + l] = ext1;
            chain();
            YF[l] = ZP_EXT[l];                               // x just above segment 0
            YL[(S - 1) * L + l] = ZP_EXT[L + l];             // x just below segment S-1
        }
        __syncthreads();
        apply(true);
    }
    if (MODE == 1) {
        // first and last unknown of the isolated super-segment (an end of the line needs only one of them)
        if (live && j == 0) h.HF[(size_t)K * plane + e] = y[0];
        if (live && j == S - 1) h.HL[(size_t)K * plane + e] = mirror ? y[0] : y[R - 1];
        return;
    }
    if (!pin) {
        // recompute the row addresses instead of keeping the R load addresses alive (registers)
        double *out0 = row0;
        ptrdiff_t ostep = step;
        asm volatile("" : "+l"(out0), "+l"(ostep));
#pragma unroll
        for (int i = 0; i < R; ++i) __stcs(out0 + i * ostep, y[i]);
    }
    // the warp that owns element 0 solves the singular line together (its line was never stored above)
    // (long lines: zero_mode_long_kernel does it with a whole CTA)
    if (MODE == 0 && p.singular && blockIdx.x == 0 && threadIdx.x < 32) zero_mode_line(w, plane, p.nz, p.bcz, p.scale, p.zero_scratch + (size_t)blockIdx.y * p.nz, p.singular == 2);
}

// Couples the super-segments of every line (see ZHier): one thread per mode.  The super-segment block
// is the rows x rows Toeplitz block; its couplings are ratios and products of its Thomas pivots
// g_k = 1 / (d_k - g_{k-1}) (no minors here: q_rows would overflow for rows = 256):
//   a1 = g_{rows-1} (interior block),  a0 = g_{rows-1} (end block, d_0 = b_end),  b1 = -prod_k g_k.
// Same interface system and the same Moebius form of its factorisation as inside the CTA.
// In: HF[K], HL[K] = first / last unknown of the isolated super-segment K.
// Out: HL[K] = x of the last row of super-segment K (K < nK-1), HF[K] = x of the first row of
// super-segment K (K > 0).  SC, SA: [nK][plane] scratch.
__global__ void __launch_bounds__(64)
zsolve_hier_interface_kernel(ZParams p, ZHier h, int rows, double *SC, double *SA) {
    const size_t plane = (size_t)p.nx * p.ny;
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= plane || (p.singular && e == 0)) return;
    const double s = p.sx[e % p.nx] + p.sy[e / p.nx];
    const double bint = -2.0 + s;
    const double bend = ((p.bcz == 1) ? -1.0 : -3.0) + s;
    // pivots of the super-segment block from its leading minors (one FMA per row), renormalised every
    // 32 rows so that nothing overflows:  g_{rows-1} = q_{rows-1} / q_rows,  prod_k g_k = 1 / q_rows
    double im = 1.0, ic = bint, em = 1.0, ec = bend, prod = 1.0;
    for (int k0 = 1; k0 < rows; k0 += 32) {
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            if (k0 + k < rows) {
                const double in = fma(bint, ic, -im), en = fma(bint, ec, -em);
                im = ic; ic = in;
                em = ec; ec = en;
            }
        }
        const double ri = fast_rcp(ic), re = fast_rcp(ec);
        prod *= ri;                       // underflows to 0 for strongly dominant modes: the coupling is 0 then
        im *= ri; ic = 1.0;
        em *= re; ec = 1.0;
    }
    const double a0 = em, a1 = im, b1 = -prod;
    const int nK = h.nK;
    const double k1 = fma(b1, b1, -a1 * a1);
    double N = a0, M = 1.0, pa = 0.0;
    constexpr int CH = 8;                 // interface values are fetched CH steps at a time (the loop is latency bound)
    for (int J0 = 0; J0 < nK - 1; J0 += CH) {
        double yl[CH], yf[CH];
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            const int J = min(J0 + i, nK - 2);
            yl[i] = h.HL[(size_t)J * plane + e];
            yf[i] = h.HF[(size_t)(J + 1) * plane + e];
        }
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            const int J = J0 + i;
            if (J < nK - 1) {
                const double vL = (J == 0) ? 0.0 : b1;
                const double vF = (J + 1 == nK - 1) ? a0 : a1, wF = (J + 1 == nK - 1) ? 0.0 : b1;
                const double r = fast_rcp(fma(-vF, N, M));
                const double D = M * r, AD = N * r;
                const double Ya = fma(-vL, pa, yl[i]);
                const double t = fma(-vF, Ya, yf[i]);
                pa = fma(-AD, t, Ya);
                h.HF[(size_t)(J + 1) * plane + e] = D * t;          // pc_J
                h.HL[(size_t)J * plane + e] = pa;                   // pa_J
                SC[(size_t)J * plane + e] = D * wF;
                SA[(size_t)J * plane + e] = -AD * wF;
                const double Nn = fma(k1, N, a1 * M), Mn = fma(-a1, N, M);
                // keep the pair (N, M) near 1: only its ratio matters
                const double nrm = fast_rcp(fabs(Mn) > fabs(Nn) ? Mn : Nn);
                N = Nn * nrm;
                M = Mn * nrm;
            }
        }
    }
    double cn = 0.0;
    for (int J0 = nK - 2; J0 >= 0; J0 -= CH) {
        double sc[CH], sa[CH], pc[CH], pv[CH];
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            const int J = max(J0 - i, 0);
            sc[i] = SC[(size_t)J * plane + e];
            sa[i] = SA[(size_t)J * plane + e];
            pc[i] = h.HF[(size_t)(J + 1) * plane + e];
            pv[i] = h.HL[(size_t)J * plane + e];
        }
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            const int J = J0 - i;
            if (J >= 0) {
                const double cv = fma(-sc[i], cn, pc[i]);
                const double av = fma(-sa[i], cn, pv[i]);
                h.HF[(size_t)(J + 1) * plane + e] = cv;             // first row of super-segment J+1
                h.HL[(size_t)J * plane + e] = av;                   // last row of super-segment J
                cn = cv;
            }
        }
    }
}

// Periodic z on two levels: every super-segment is an interior block and the chain of nK interfaces closes on
// itself.  Same treatment as inside the CTA (zsolve_part_kernel, CYC): the open chain is factored and solved for
// the right-hand side and for the two unit vectors of the wrap-around couplings (z1 = chain^-1 e(row a_0),
// z2 = chain^-1 e(row c_{nK-1})), and a 2x2 closure gives the wrapped unknowns -- an exact cyclic solve, in place
// of Sherman-Morrison's second sweep over the whole line.
// In / out as zsolve_hier_interface_kernel, with K + 1 and K - 1 taken modulo nK.  W: [6][nK][plane] scratch.
__global__ void __launch_bounds__(64)
zsolve_hier_interface_cyclic_kernel(ZParams p, ZHier h, int rows, double *W) {
    const size_t plane = (size_t)p.nx * p.ny;
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= plane || (p.singular && e == 0)) return;
    const double s = p.sx[e % p.nx] + p.sy[e / p.nx];
    const double bint = -2.0 + s;
    double im = 1.0, ic = bint, prod = 1.0;
    for (int k0 = 0; k0 + 1 < rows; k0 += 31) {       // 31 steps per renormalisation: |minor| <= bmax^32 (zpart_range_ok)
#pragma unroll
        for (int k = 1; k <= 31; ++k) {
            if (k0 + k < rows) {
                const double in = fma(bint, ic, -im);
                im = ic; ic = in;
            }
        }
        const double ri = fast_rcp(ic);
        prod *= ri;
        im *= ri; ic = 1.0;
    }
    const double a1 = im, b1 = -prod;
    const int nK = h.nK;
    const size_t slab = (size_t)nK * plane;
    double *SC = W + e, *SA = SC + slab, *Z1C = SA + slab, *Z1A = Z1C + slab, *Z2C = Z1A + slab, *Z2A = Z2C + slab;
    double *HF = h.HF + e, *HL = h.HL + e;
    const double k1 = fma(b1, b1, -a1 * a1);
    constexpr int CH = 8;                 // values are fetched CH steps at a time (the loops are latency bound)
    {
        double N = a1, M = 1.0, pa = 0.0, pa1 = 0.0;
        for (int J0 = 0; J0 < nK; J0 += CH) {
            double yl[CH], yf[CH];
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                const int J = min(J0 + i, nK - 1);
                yl[i] = HL[(size_t)J * plane];
                yf[i] = HF[(size_t)((J + 1 < nK) ? J + 1 : 0) * plane];
            }
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                const int J = J0 + i;
                if (J < nK) {
                    const int JF = (J + 1 < nK) ? J + 1 : 0;
                    const double vL = (J == 0) ? 0.0 : b1, wF = (J == nK - 1) ? 0.0 : b1;
                    const double r = fast_rcp(fma(-a1, N, M));
                    const double D = M * r, AD = N * r;
                    const double Ya = fma(-vL, pa, yl[i]);
                    const double t = fma(-a1, Ya, yf[i]);
                    pa = fma(-AD, t, Ya);
                    const double Ya1 = fma(-vL, pa1, (J == 0) ? 1.0 : 0.0);
                    const double t1 = -a1 * Ya1;
                    pa1 = fma(-AD, t1, Ya1);
                    HF[(size_t)JF * plane] = D * t;                 // pc_J
                    HL[(size_t)J * plane] = pa;                     // pa_J
                    SC[(size_t)J * plane] = D * wF;
                    SA[(size_t)J * plane] = -AD * wF;
                    Z1C[(size_t)J * plane] = D * t1;
                    Z1A[(size_t)J * plane] = pa1;
                    Z2C[(size_t)J * plane] = (J == nK - 1) ? D : 0.0;
                    Z2A[(size_t)J * plane] = (J == nK - 1) ? -AD : 0.0;
                    const double Nn = fma(k1, N, a1 * M), Mn = fma(-a1, N, M);
                    const double nrm = fast_rcp(fabs(Mn) > fabs(Nn) ? Mn : Nn);
                    N = Nn * nrm;
                    M = Mn * nrm;
                }
            }
        }
    }
    double z1a_last = 0.0, z2a_last = 0.0, z1c_0 = 0.0, z2c_0 = 0.0, x0a = 0.0, x0c = 0.0;
    {
        double cn = 0.0, c1 = 0.0, c2 = 0.0;
        for (int J0 = nK - 1; J0 >= 0; J0 -= CH) {
            double sc[CH], sa[CH], pc[CH], pv[CH], u1c[CH], u1a[CH], u2c[CH], u2a[CH];
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                const int J = max(J0 - i, 0);
                sc[i] = SC[(size_t)J * plane];
                sa[i] = SA[(size_t)J * plane];
                pc[i] = HF[(size_t)((J + 1 < nK) ? J + 1 : 0) * plane];
                pv[i] = HL[(size_t)J * plane];
                u1c[i] = Z1C[(size_t)J * plane]; u1a[i] = Z1A[(size_t)J * plane];
                u2c[i] = Z2C[(size_t)J * plane]; u2a[i] = Z2A[(size_t)J * plane];
            }
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                const int J = J0 - i;
                if (J >= 0) {
                    const int JF = (J + 1 < nK) ? J + 1 : 0;
                    const double av = fma(-sa[i], cn, pv[i]), a1v = fma(-sa[i], c1, u1a[i]), a2v = fma(-sa[i], c2, u2a[i]);
                    cn = fma(-sc[i], cn, pc[i]);
                    c1 = fma(-sc[i], c1, u1c[i]);
                    c2 = fma(-sc[i], c2, u2c[i]);
                    HF[(size_t)JF * plane] = cn;                    // open-chain c_J
                    HL[(size_t)J * plane] = av;                     // open-chain a_J
                    Z1C[(size_t)J * plane] = c1; Z1A[(size_t)J * plane] = a1v;
                    Z2C[(size_t)J * plane] = c2; Z2A[(size_t)J * plane] = a2v;
                    if (J == nK - 1) { z1a_last = a1v; z2a_last = a2v; x0a = av; }
                    if (J == 0) { z1c_0 = c1; z2c_0 = c2; x0c = cn; }
                }
            }
        }
    }
    // closure:  K (a_{nK-1}, c_0)^T = (x0a, x0c)^T,  K = [1 + b1 z1a_{nK-1}, b1 z2a_{nK-1}; b1 z1c_0, 1 + b1 z2c_0];
    //           x = x0 - (b1 a_{nK-1}) z1 - (b1 c_0) z2
    const double k11 = fma(b1, z1a_last, 1.0), k12 = b1 * z2a_last, k21 = b1 * z1c_0, k22 = fma(b1, z2c_0, 1.0);
    const double rdet = b1 / fma(k11, k22, -k12 * k21);
    const double ba = (k22 * x0a - k12 * x0c) * rdet, bg = (k11 * x0c - k21 * x0a) * rdet;
    for (int J = 0; J < nK; ++J) {
        const int JF = (J + 1 < nK) ? J + 1 : 0;
        HF[(size_t)JF * plane] = fma(-ba, Z1C[(size_t)J * plane], fma(-bg, Z2C[(size_t)J * plane], HF[(size_t)JF * plane]));
        HL[(size_t)J * plane] = fma(-ba, Z1A[(size_t)J * plane], fma(-bg, Z2A[(size_t)J * plane], HL[(size_t)J * plane]));
    }
}

// The singular (0,0) line of a long Neumann- or periodic-z problem (R11), by one CTA of
// 1024 threads: the same two running sums as zero_mode_line, each thread holding its contiguous
// chunk of at most 16 rows in registers (nz <= 16384), chunk totals combined by block-wide scans.
//   r <- (r - mean r) scale;  x_0 = 0;  d_k = -sum_{m >= k} r_m  (periodic: d_1 + sum_{1 <= m < k} r_m);
//   x_k = sum_{1 <= m <= k} d_m;  x <- x - mean x
__device__ __forceinline__ double zp_block_excl_scan(double v, double *red, double &total) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const double wex = warp_excl_scan(v, lane);
    const double wtot = __shfl_sync(0xffffffffu, wex + v, 31);
    __syncthreads();                                          // red may still be read from the previous call
    if (lane == 0) red[wid] = wtot;
    __syncthreads();
    const double mine = (lane < nw) ? red[lane] : 0.0;
    const double wprefix = warp_excl_scan(mine, lane);
    total = __shfl_sync(0xffffffffu, wprefix + mine, 31);
    return __shfl_sync(0xffffffffu, wprefix, wid) + wex;
}

__global__ void __launch_bounds__(1024, 1)
zero_mode_long_kernel(double *col, size_t plane, int nz, double scale, int pin_plane0, int periodic) {
    __shared__ double red[32];
    constexpr int C = 16;
    const int c = (nz + (int)blockDim.x - 1) / (int)blockDim.x;        // <= C
    const int k0 = min((int)threadIdx.x * c, nz), k1 = min(k0 + c, nz);
    double v[C];
    double acc = 0.0, tot;
#pragma unroll
    for (int i = 0; i < C; ++i) {
        v[i] = (i < c && k0 + i < k1) ? col[(size_t)(k0 + i) * plane] * scale : 0.0;
        acc += v[i];
    }
    zp_block_excl_scan(acc, red, tot);
    const double mean = tot / nz;
    // rows >= 1 only; v <- r - mean
    double own = 0.0;
#pragma unroll
    for (int i = 0; i < C; ++i) {
        const bool in = i < c && k0 + i < k1 && k0 + i >= 1;
        v[i] = in ? v[i] - mean : 0.0;
        own += v[i];
    }
    double all;
    double run = zp_block_excl_scan(own, red, all);
    double dsum = 0.0;
    if (!periodic) {
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const bool in = i < c && k0 + i < k1 && k0 + i >= 1;
            const double r = v[i];
            v[i] = in ? -(all - run) : 0.0;                           // Neumann: d_k = -sum_{m >= k} r_m
            run += r;
            dsum += v[i];
        }
    } else {
        // periodic: d_k = d_1 + S_{k-1}, S_j = sum_{1 <= m <= j} r_m, and x_n = x_0 = 0 fixes d_1 = -(sum_k S_{k-1} + S_{n-1}) / n
        double ssum = 0.0;
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const bool in = i < c && k0 + i < k1 && k0 + i >= 1;
            const double r = v[i];
            v[i] = in ? run : 0.0;                                    // S_{k-1}
            run += r;
            ssum += v[i];
        }
        double stot;
        zp_block_excl_scan(ssum, red, stot);
        const double d1 = -(stot + all) / nz;
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const bool in = i < c && k0 + i < k1 && k0 + i >= 1;
            v[i] = in ? v[i] + d1 : 0.0;
            dsum += v[i];
        }
    }
    double dummy;
    double x = zp_block_excl_scan(dsum, red, dummy);
    double xs = 0.0;
#pragma unroll
    for (int i = 0; i < C; ++i) {
        x += v[i];
        v[i] = x;                                                     // x_k (x_0 = 0)
        if (i < c && k0 + i < k1) xs += x;
    }
    double xtot;
    zp_block_excl_scan(xs, red, xtot);
    const double xmean = pin_plane0 ? 0.0 : xtot / nz;
#pragma unroll
    for (int i = 0; i < C; ++i)
        if (i < c && k0 + i < k1) col[(size_t)(k0 + i) * plane] = v[i] - xmean;
}

}  // namespace pp
