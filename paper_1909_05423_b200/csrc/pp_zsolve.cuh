// z-solve kernels: one tridiagonal system in z per (kx, ky), Thomas algorithm
// specialised to the Toeplitz coefficients of Algorithm 2: three values per
// diagonal (first / interior / last row), nothing N-sized stored besides the right-hand side.
//
// "Two-dimensional batch" mode: threads run across (kx, ky) -- consecutive threads
// own consecutive x positions, so every z step of the sweep is one coalesced plane-row access.
// After the x/y passes every real element of a plane is an independent real system (Re and Im of a
// complex mode share the real matrix), with shift
//     s = dz^2 (lam_x/dx^2 + lam_y/dy^2)                               (Table 2)
// read from two small per-axis tables.  T = L_z + s I:
//     interior diagonal -2 + s, off-diagonals 1, first/last diagonal -1 + s (Neumann) / -3 + s
//     (Dirichlet); periodic: cyclic corners, solved by Sherman-Morrison.
//
// Recurrence (Algorithm 1, with g_k = 1/beta_k; g_{-1} = x'_{-1} = 0):
//     g_k  = 1 / (b_k - g_{k-1}),   x'_k = (r_k - x'_{k-1}) g_k          forward
//     x_k  = x'_k - g_k x_{k+1}                                          backward
// The pivots g_k are not stored (the paper's gamma[N] container): the forward sweep keeps one
// checkpoint every CB rows and the backward sweep recomputes each block of CB pivots from its
// checkpoint, bit-identically, in registers.
//
// The (0,0) system of an all-periodic/Neumann problem is singular: its line is left
// untouched by the main sweeps and solved by `zero_mode_line` (mean-projected right-hand side,
// x_0 pinned, zero-mean result).
#pragma once
#include <cuda_runtime.h>

#include "pp_zshape.h"

namespace pp {

struct ZParams {
    int nx, ny, nz;
    int bcz;
    int singular;            // 1, 2: element 0 (kx = ky = 0) is the singular zero mode; 2: return the solution whose
                             // z = 0 plane has zero mean (the paper's default) instead of zero volume mean
    double scale;            // dz^2 / (nx ny): rhs scaling incl. the inverse-transform normalisation
    const double *sx;        // [nx]  dz^2 lam_x(kx(ix)) / dx^2
    const double *sy;        // [ny]  dz^2 lam_y(ky(j))  / dy^2
    double *zero_scratch;    // [Z_MAX_BATCH][nz]  scratch lines for the zero-mode solve
    size_t batch_stride;     // one-CTA partitioned kernel, pp_solve_batch: blockIdx.y selects the grid, this many doubles apart
};


// L2 eviction-priority hints (createpolicy + .L2::cache_hint).  The forward sweep's x' values are
// re-read by the backward sweep: they are stored "evict_last" so they survive in the 126 MB L2,
// while the streams that are touched once (right-hand side in, solution out) are "evict_first".
#ifndef PP_Z_HINTS
#define PP_Z_HINTS 1
#endif
#ifndef PP_Z_THREADS
#define PP_Z_THREADS 256
#endif
#ifndef PP_Z_MINB
#define PP_Z_MINB 2
#endif
struct ZPolicy {
    unsigned long long first, last;
    __device__ __forceinline__ ZPolicy() {
#if PP_Z_HINTS
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(first));
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(last));
#else
        first = last = 0;
#endif
    }
};
__device__ __forceinline__ double ld_hint(const double *p, unsigned long long pol) {
#if PP_Z_HINTS
    double v;
    asm volatile("ld.global.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
    return v;
#else
    return *p;
#endif
}
__device__ __forceinline__ void st_hint(double *p, double v, unsigned long long pol) {
#if PP_Z_HINTS
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
#else
    *p = v;
#endif
}

// The singular (0,0) line, solved cooperatively by one full warp (R11):
//   r <- (r - mean r) * scale;  pin x_0 = 0 and drop row 0;  solve rows 1..nz-1 of L_z;  x <- x - mean x.
// With s = 0 the rows are pure second differences, so the pinned system is solved by two running
// sums instead of a serial elimination (d_k = x_k - x_{k-1}):
//   Neumann :  d_k = -sum_{m >= k} r_m                      (last row: x_{n-2} - x_{n-1} = r_{n-1})
//   periodic:  d_k = d_1 + sum_{1 <= m < k} r_m,  d_1 fixed by x_n = x_0 = 0
//   x_k = sum_{1 <= m <= k} d_m.
// Each lane scans a contiguous chunk; chunk totals are combined with warp shuffles.  `tmp` is a
// plan-owned scratch line of nz doubles.  All 32 lanes must call this.
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// exclusive prefix of per-lane totals (lane order ascending)
__device__ __forceinline__ double warp_excl_scan(double v, int lane) {
    double inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    return inc - v;
}

__device__ __noinline__ void zero_mode_line(double *col, size_t plane, int nz, int bcz, double scale, double *tmp,
                                            bool pin_plane0) {
    const int lane = threadIdx.x & 31;
    const int c = (nz + 31) / 32;
    const int k0 = min(lane * c, nz), k1 = min(k0 + c, nz);
    // mean of r
    double acc = 0.0;
    for (int k = k0; k < k1; ++k) { const double r = col[(size_t)k * plane] * scale; tmp[k] = r; acc += r; }
    const double mean = warp_sum(acc) / nz;
    // running sums of (r - mean) over rows 1..nz-1  ->  d_k in tmp[k]
    double tot = 0.0;
    for (int k = max(k0, 1); k < k1; ++k) tot += tmp[k] - mean;
    const double before = warp_excl_scan(tot, lane);          // sum over lanes below
    const double all = __shfl_sync(0xffffffffu, before + tot, 31);
    __syncwarp();
    if (bcz == 1) {
        // Neumann: d_k = -(sum_{m >= k} r_m) = -(all - sum_{m < k} r_m)
        double run = before;
        for (int k = max(k0, 1); k < k1; ++k) { const double r = tmp[k] - mean; tmp[k] = -(all - run); run += r; }
    } else {
        // periodic: d_k = d_1 + S_{k-1}, S_j = sum_{1 <= m <= j} r_m; first store S_{k-1}, then add d_1
        double run = before;
        for (int k = max(k0, 1); k < k1; ++k) { const double r = tmp[k] - mean; tmp[k] = run; run += r; }
        // x_n = 0:  n d_1 + sum_{k=1..n} S_{k-1} = 0, S_{n-1} = all
        double ssum = 0.0;
        for (int k = max(k0, 1); k < k1; ++k) ssum += tmp[k];
        const double d1 = -(warp_sum(ssum) + all) / nz;
        for (int k = max(k0, 1); k < k1; ++k) tmp[k] += d1;
    }
    __syncwarp();
    // x_k = sum_{1 <= m <= k} d_m
    double dt = 0.0;
    for (int k = max(k0, 1); k < k1; ++k) dt += tmp[k];
    double run = warp_excl_scan(dt, lane);
    double xs = 0.0;
    for (int k = max(k0, 1); k < k1; ++k) { run += tmp[k]; tmp[k] = run; xs += run; }
    // x_0 = 0 contributes nothing; with the plane-0 convention the pinned x_0 = 0 already is the answer
    const double xmean = pin_plane0 ? 0.0 : warp_sum(xs) / nz;
    for (int k = k0; k < k1; ++k) col[(size_t)k * plane] = ((k == 0) ? 0.0 : tmp[k]) - xmean;
}

// Reciprocal to ~1 ulp: MUFU.RCP64H seed (>= 20 bits) + two Newton steps.  The operands here are
// pivot products |q| >= 1 of a diagonally dominant matrix -- never zero, subnormal or infinite.
__device__ __forceinline__ double fast_rcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    return r;
}

// Neumann / Dirichlet in z.  One thread per real element of a plane; block of TH threads.
//
// Division-free sweeps.  Inside a block of CB rows starting at k0 the pivots are carried as the
// ratio g_k = q_i / q_{i+1} (k = k0 + i) of the three-term recurrence
//     q_{-1} = g_{k0-1},  q_0 = 1,  q_{i+1} = b_k q_i - q_{i-1}
// and the eliminated right-hand side as y_i = x'_k q_{i+1}:
//     y_i = r_k q_i - y_{i-1}                                   (y_{-1} = x'_{k0-1})
// -- one dependent FMA per row on each chain instead of a dependent division.  The forward sweep
// stores y_i and renormalises (one reciprocal) at the end of every block, where it also leaves the
// checkpoint g_{k0-1} in shared memory; |q| grows by at most |b|^CB inside a block.  The backward
// sweep recomputes the block's q_i bit-identically from the checkpoint and substitutes
//     x_k = (y_i - q_i x_{k+1}) / q_{i+1},
// whose reciprocals are off the dependency chain.
//
// Two-sided elimination.  T is persymmetric (same first and last diagonal), so eliminating upwards
// from the last row produces the same pivots as eliminating downwards from the first.  Each thread
// therefore runs both at once -- rows kk and nz-1-kk, kk = 0 .. ceil(nz/2)-1, share one pivot chain
// and give two independent right-hand-side chains and twice the loads in flight -- couples the two
// halves in the middle with a 2x2 solve, and substitutes outwards in both directions.  Half the
// pivot arithmetic, and the same memory-level parallelism from half as many resident threads, which
// keeps the forward sweep's output in L2 until the backward sweep re-reads it.
template <int CB, bool FIRST>
__device__ __forceinline__ void z_block_pivots(double (&qq)[CB + 1], double qm, double bint, double bend) {
    qq[0] = 1.0;
#pragma unroll
    for (int i = 0; i < CB; ++i) {
        const double bk = (FIRST && i == 0) ? bend : bint;
        qq[i + 1] = fma(bk, qq[i], -qm);
        qm = qq[i];
    }
}

struct ZHalfState {
    double g, xt, xb;          // normalised carries: pivot ratio, x' of the top chain, x' of the bottom chain
    double qcap, qmcap, ycap;  // bottom chain's state at its last row (only when it ends before the top chain)
};

// rows kk = k0 .. k0+CB-1 of both halves.  m = rows of the top half, nb = rows of the bottom half.
template <int CB, bool FIRST, bool RAGGED>
__device__ __forceinline__ void z_forward_block(double *top, double *bot, ptrdiff_t plane, int k0, int m, int nb,
                                                double bint, double bend, double scale, bool pin,
                                                const ZPolicy &pol, ZHalfState &st) {
    double rt[CB], rb[CB];
#pragma unroll
    for (int i = 0; i < CB; ++i) {
        const int kk = k0 + i;
        rt[i] = (!RAGGED || kk < m) ? ld_hint(top + kk * plane, pol.first) : 0.0;
        rb[i] = (!RAGGED || kk < nb) ? ld_hint(bot - kk * plane, pol.first) : 0.0;
    }
    double qm = st.g, q = 1.0, yt = st.xt, yb = st.xb;
#pragma unroll
    for (int i = 0; i < CB; ++i) {
        const int kk = k0 + i;
        if (!RAGGED || kk < m) {
            const double bk = (FIRST && i == 0) ? bend : bint;
            yt = fma(rt[i] * scale, q, -yt);
            if (!pin) st_hint(top + kk * plane, yt, pol.last);
            if (!RAGGED || kk < nb) {
                yb = fma(rb[i] * scale, q, -yb);
                if (!pin) st_hint(bot - kk * plane, yb, pol.last);
            }
            const double qn = fma(bk, q, -qm);
            qm = q;
            q = qn;
            if (RAGGED && kk == nb - 1) { st.qcap = q; st.qmcap = qm; st.ycap = yb; }
        }
    }
    const double rq = fast_rcp(q);
    st.g = qm * rq;
    st.xt = yt * rq;
    st.xb = yb * rq;
}

template <int CB, bool FIRST, bool RAGGED>
__device__ __forceinline__ void z_backward_block(double *top, double *bot, ptrdiff_t plane, int k0, int m, int nb,
                                                 double gprev, double bint, double bend, bool pin,
                                                 const ZPolicy &pol, double &xt, double &xb) {
    double qq[CB + 1], yt[CB], yb[CB];
#pragma unroll
    for (int i = 0; i < CB; ++i) {
        const int kk = k0 + i;
        yt[i] = (!RAGGED || kk < m) ? ld_hint(top + kk * plane, pol.first) : 0.0;
        yb[i] = (!RAGGED || kk < nb) ? ld_hint(bot - kk * plane, pol.first) : 0.0;
    }
    z_block_pivots<CB, FIRST>(qq, gprev, bint, bend);
#pragma unroll
    for (int i = CB - 1; i >= 0; --i) {
        const int kk = k0 + i;
        if (!RAGGED || kk < m) {
            const double rq = fast_rcp(qq[i + 1]);
            const double c = qq[i] * rq;
            xt = fma(-c, xt, yt[i] * rq);
            if (!pin) st_hint(top + kk * plane, xt, pol.first);
            if (!RAGGED || kk < nb) {
                xb = fma(-c, xb, yb[i] * rq);
                if (!pin) st_hint(bot - kk * plane, xb, pol.first);
            }
        }
    }
}

template <int CB, int TH>
__global__ void __launch_bounds__(TH, PP_Z_MINB)
zsolve_thomas_kernel(double *w, ZParams p) {
    extern __shared__ double ck[];                            // [nblk][TH] checkpoints g_{k0-1}
    const size_t plane = (size_t)p.nx * p.ny;
    const size_t e = (size_t)blockIdx.x * TH + threadIdx.x;
    const bool live = e < plane;                              // dead threads run along (warp-wide zero-mode solve) but never store
    const int ix = live ? (int)(e % p.nx) : 0, j = live ? (int)(e / p.nx) : 0;
    const bool pin = !live || (p.singular && e == 0);
    const double s = pin ? -1.0 : (p.sx[ix] + p.sy[j]);      // pinned line: placeholder, results discarded
    const double bint = -2.0 + s;
    const double bend = ((p.bcz == 1) ? -1.0 : -3.0) + s;
    const int nz = p.nz;
    const int m = (nz + 1) / 2, nb = nz - m;                  // top rows [0, m), bottom rows nz-1-kk, kk in [0, nb)
    const int nblk = (m + CB - 1) / CB;
    const double scale = p.scale;
    const ptrdiff_t pl = (ptrdiff_t)plane;
    double *top = w + (live ? e : 0);
    double *bot = top + (ptrdiff_t)(nz - 1) * pl;
    const ZPolicy pol;
    double *myck = ck + threadIdx.x;

    // forward elimination from both ends
    ZHalfState st = {0.0, 0.0, 0.0, 1.0, 0.0, 0.0};
    for (int b = 0; b < nblk; ++b) {
        const int k0 = b * CB;
        myck[b * TH] = st.g;
        const bool ragged = (k0 + CB > m) || (nb != m && k0 + CB >= nb);   // guards, and the bottom chain's last row
        if (b == 0) {
            if (ragged) z_forward_block<CB, true, true>(top, bot, pl, k0, m, nb, bint, bend, scale, pin, pol, st);
            else        z_forward_block<CB, true, false>(top, bot, pl, k0, m, nb, bint, bend, scale, pin, pol, st);
        } else {
            if (ragged) z_forward_block<CB, false, true>(top, bot, pl, k0, m, nb, bint, bend, scale, pin, pol, st);
            else        z_forward_block<CB, false, false>(top, bot, pl, k0, m, nb, bint, bend, scale, pin, pol, st);
        }
    }
    // couple the halves:  x_{m-1} + g_t x_m = x'_t,   x_m + g_b x_{m-1} = x'_b
    double gb = st.g, xpb = st.xb;
    if (nb != m) {                                            // odd nz: the bottom chain ended one row earlier
        const double rqc = fast_rcp(st.qcap);
        gb = st.qmcap * rqc;
        xpb = st.ycap * rqc;
    }
    const double rden = 1.0 / (1.0 - st.g * gb);
    double xt = (xpb - gb * st.xt) * rden;                    // x_m     : the row after the top half's last
    double xb = (st.xt - st.g * xpb) * rden;                  // x_{m-1} : the row after the bottom half's last
    // back substitution outwards
    for (int b = nblk - 1; b >= 0; --b) {
        const int k0 = b * CB;
        const double gprev = myck[b * TH];
        const bool ragged = (k0 + CB > m) || (nb != m && k0 + CB >= nb);   // guards, and the bottom chain's last row
        if (b == 0) {
            if (ragged) z_backward_block<CB, true, true>(top, bot, pl, k0, m, nb, gprev, bint, bend, pin, pol, xt, xb);
            else        z_backward_block<CB, true, false>(top, bot, pl, k0, m, nb, gprev, bint, bend, pin, pol, xt, xb);
        } else {
            if (ragged) z_backward_block<CB, false, true>(top, bot, pl, k0, m, nb, gprev, bint, bend, pin, pol, xt, xb);
            else        z_backward_block<CB, false, false>(top, bot, pl, k0, m, nb, gprev, bint, bend, pin, pol, xt, xb);
        }
    }
    // the warp that owns element 0 solves the singular line together (block 0, warp 0: all lanes alive)
    if (p.singular && e < 32) zero_mode_line(w, plane, nz, p.bcz, scale, p.zero_scratch, p.singular == 2);
}

// Periodic in z: Sherman-Morrison, "two solves".  With gamma = -b:
//   T' = T - w v^T,  w = (gamma,0,..,0,1)^T, v = (1,0,..,0,1/gamma)^T,  b'_0 = 2b, b'_{n-1} = b + 1/b
//   x = T'^-1 r,  q = T'^-1 w,  u = x - q (v.x)/(1 + v.q).
// q depends only on the mode, so it is never stored: it is recomputed next to the pivots, from checkpoints
// kept every CB rows in shared memory.
// Sweep 1 forward (x'), sweep 2 backward (x, and q to get the scalar), sweep 3 backward (u).
template <int CB, int TH>
__global__ void __launch_bounds__(TH, PP_Z_MINB)
zsolve_cyclic_kernel(double *w, ZParams p) {
    extern __shared__ double ck[];                 // [2][nblk][TH] checkpoints of the pivot and of the q sweep
    const size_t plane = (size_t)p.nx * p.ny;
    const size_t e = (size_t)blockIdx.x * TH + threadIdx.x;
    const bool live = e < plane;
    const int ix = live ? (int)(e % p.nx) : 0, j = live ? (int)(e / p.nx) : 0;
    const bool pin = !live || (p.singular && e == 0);
    const double s = pin ? -1.0 : (p.sx[ix] + p.sy[j]);
    const double b = -2.0 + s;
    const double gamma = -b;
    const double bfirst = b - gamma;              // 2b
    const double blast = b - 1.0 / gamma;         // b + 1/b
    const int nz = p.nz;
    const double scale = p.scale;
    double *col = w + (live ? e : 0);
    const ZPolicy pol;
    const int nblk = (nz + CB - 1) / CB;
    double *ckg = ck + threadIdx.x, *ckq = ckg + (size_t)nblk * TH;     // entry of block i at [i * TH]

    double g = 0.0, xp = 0.0, qp = 0.0;
    for (int k0 = 0; k0 < nz; k0 += CB) {
        ckg[(k0 / CB) * TH] = g;
        ckq[(k0 / CB) * TH] = qp;
        double r[CB];
#pragma unroll
        for (int i = 0; i < CB; ++i) r[i] = (k0 + i < nz) ? ld_hint(col + (size_t)(k0 + i) * plane, pol.first) : 0.0;
#pragma unroll
        for (int i = 0; i < CB; ++i) {
            const int k = k0 + i;
            if (k < nz) {
                const double bk = (k == 0) ? bfirst : ((k == nz - 1) ? blast : b);
                const double wk = (k == 0) ? gamma : ((k == nz - 1) ? 1.0 : 0.0);
                g = 1.0 / (bk - g);
                xp = (r[i] * scale - xp) * g;
                qp = (wk - qp) * g;
                if (!pin) st_hint(col + (size_t)k * plane, xp, pol.last);
            }
        }
    }
    const double xlast = xp, qlast = qp;
    double fac = 0.0;
    for (int sweep = 0; sweep < 2; ++sweep) {
        double x = xlast, q = qlast;
        if (sweep == 1 && !pin) col[(size_t)(nz - 1) * plane] = xlast - fac * qlast;
        for (int k0 = ((nz - 1) / CB) * CB; k0 >= 0; k0 -= CB) {
            double gl[CB], ql[CB], r[CB];
            double gg = ckg[(k0 / CB) * TH], qq = ckq[(k0 / CB) * TH];
#pragma unroll
            for (int i = 0; i < CB; ++i) r[i] = (k0 + i < nz - 1) ? ld_hint(col + (size_t)(k0 + i) * plane, sweep == 0 ? pol.last : pol.first) : 0.0;
#pragma unroll
            for (int i = 0; i < CB; ++i) {
                const int k = k0 + i;
                const double bk = (k == 0) ? bfirst : ((k == nz - 1) ? blast : b);
                const double wk = (k == 0) ? gamma : ((k == nz - 1) ? 1.0 : 0.0);
                gg = 1.0 / (bk - gg);
                qq = (wk - qq) * gg;
                gl[i] = gg;
                ql[i] = qq;
            }
#pragma unroll
            for (int i = CB - 1; i >= 0; --i) {
                const int k = k0 + i;
                if (k < nz - 1) {
                    q = ql[i] - gl[i] * q;
                    if (sweep == 0) {
                        x = r[i] - gl[i] * x;                  // r holds x'_k
                        if (!pin) st_hint(col + (size_t)k * plane, x, pol.last);
                    } else {
                        if (!pin) st_hint(col + (size_t)k * plane, r[i] - fac * q, pol.first);   // r holds x_k
                    }
                }
            }
        }
        if (sweep == 0) fac = (x + xlast / gamma) / (1.0 + q + qlast / gamma);
    }
    // the warp that owns element 0 solves the singular line together (block 0, warp 0: all lanes alive)
    if (p.singular && e < 32) zero_mode_line(w, plane, nz, p.bcz, scale, p.zero_scratch, p.singular == 2);
}

}  // namespace pp
