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

namespace pp {

struct ZParams {
    int nx, ny, nz;
    int bcz;
    int singular;            // 1: element 0 (kx = ky = 0) is the singular zero mode
    double scale;            // dz^2 / (nx ny): rhs scaling incl. the inverse-transform normalisation
    const double *sx;        // [nx]  dz^2 lam_x(kx(ix)) / dx^2
    const double *sy;        // [ny]  dz^2 lam_y(ky(j))  / dy^2
    double *zero_scratch;    // [nz]  pivots of the zero-mode line
};

constexpr int Z_MAX_CK = 64;   // checkpoints per line

// Serial solve of the singular (0,0) line by one thread (R11):
// r <- (r - mean r) * scale; x_0 = 0; Thomas on rows 1..nz-1 of L_z; x <- x - mean x.
__device__ __noinline__ void zero_mode_line(double *col, size_t plane, int nz, int bcz, double scale, double *gam) {
    double sum = 0.0;
    for (int k = 0; k < nz; ++k) sum += col[k * plane];
    const double mean = sum / nz;
    const double blast = (bcz == 1) ? -1.0 : -2.0;     // Neumann: -1; periodic: corners dropped with row 0
    if (nz >= 2) {
        double beta = (nz == 2) ? blast : -2.0;
        double x = ((col[plane] - mean) * scale) / beta;
        col[plane] = x;
        for (int k = 2; k < nz; ++k) {
            const double g = 1.0 / beta;
            gam[k] = g;
            beta = ((k == nz - 1) ? blast : -2.0) - g;
            x = ((col[k * plane] - mean) * scale - x) / beta;
            col[k * plane] = x;
        }
        for (int k = nz - 2; k >= 1; --k) {
            x = col[k * plane] - gam[k + 1] * x;
            col[k * plane] = x;
        }
    }
    col[0] = 0.0;
    double s2 = 0.0;
    for (int k = 1; k < nz; ++k) s2 += col[k * plane];
    const double m2 = s2 / nz;
    for (int k = 0; k < nz; ++k) col[k * plane] -= m2;
}

// Neumann / Dirichlet in z.  One thread per real element of a plane.
template <int CB>
__global__ void __launch_bounds__(256)
zsolve_thomas_kernel(double *w, ZParams p) {
    const size_t plane = (size_t)p.nx * p.ny;
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= plane) return;
    const int ix = (int)(e % p.nx), j = (int)(e / p.nx);
    const bool pin = p.singular && e == 0;
    const double s = pin ? -1.0 : (p.sx[ix] + p.sy[j]);      // pinned line: placeholder, results discarded
    const double bint = -2.0 + s;
    const double bend = ((p.bcz == 1) ? -1.0 : -3.0) + s;
    const int nz = p.nz;
    const double scale = p.scale;
    double *col = w + e;
    double ck[Z_MAX_CK];

    // forward sweep, in blocks of CB rows: batch the loads, then run the chain
    double g = 0.0, xp = 0.0;
    for (int k0 = 0; k0 < nz; k0 += CB) {
        ck[k0 / CB] = g;
        double r[CB];
#pragma unroll
        for (int i = 0; i < CB; ++i) r[i] = (k0 + i < nz) ? col[(size_t)(k0 + i) * plane] : 0.0;
#pragma unroll
        for (int i = 0; i < CB; ++i) {
            const int k = k0 + i;
            if (k < nz) {
                const double bk = (k == 0 || k == nz - 1) ? bend : bint;
                g = 1.0 / (bk - g);
                xp = (r[i] * scale - xp) * g;
                if (!pin) col[(size_t)k * plane] = xp;
            }
        }
    }
    // backward sweep
    double x = xp;                                            // x_{nz-1} = x'_{nz-1}, already stored
    for (int k0 = ((nz - 1) / CB) * CB; k0 >= 0; k0 -= CB) {
        double gl[CB], r[CB];
        double gg = ck[k0 / CB];
#pragma unroll
        for (int i = 0; i < CB; ++i) r[i] = (k0 + i < nz - 1) ? col[(size_t)(k0 + i) * plane] : 0.0;
#pragma unroll
        for (int i = 0; i < CB; ++i) {
            const int k = k0 + i;
            const double bk = (k == 0 || k == nz - 1) ? bend : bint;
            gg = 1.0 / (bk - gg);
            gl[i] = gg;
        }
#pragma unroll
        for (int i = CB - 1; i >= 0; --i) {
            const int k = k0 + i;
            if (k < nz - 1) {
                x = r[i] - gl[i] * x;
                if (!pin) col[(size_t)k * plane] = x;
            }
        }
    }
    if (pin) zero_mode_line(col, plane, nz, p.bcz, scale, p.zero_scratch);
}

// Periodic in z: Sherman-Morrison, "two solves".  With gamma = -b:
//   T' = T - w v^T,  w = (gamma,0,..,0,1)^T, v = (1,0,..,0,1/gamma)^T,  b'_0 = 2b, b'_{n-1} = b + 1/b
//   x = T'^-1 r,  q = T'^-1 w,  u = x - q (v.x)/(1 + v.q).
// q depends only on the mode, so it is never stored: it is recomputed next to the pivots.
// Sweep 1 forward (x'), sweep 2 backward (x, and q to get the scalar), sweep 3 backward (u).
template <int CB>
__global__ void __launch_bounds__(256)
zsolve_cyclic_kernel(double *w, ZParams p) {
    const size_t plane = (size_t)p.nx * p.ny;
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= plane) return;
    const int ix = (int)(e % p.nx), j = (int)(e / p.nx);
    const bool pin = p.singular && e == 0;
    const double s = pin ? -1.0 : (p.sx[ix] + p.sy[j]);
    const double b = -2.0 + s;
    const double gamma = -b;
    const double bfirst = b - gamma;              // 2b
    const double blast = b - 1.0 / gamma;         // b + 1/b
    const int nz = p.nz;
    const double scale = p.scale;
    double *col = w + e;
    double ckg[Z_MAX_CK], ckq[Z_MAX_CK];

    double g = 0.0, xp = 0.0, qp = 0.0;
    for (int k0 = 0; k0 < nz; k0 += CB) {
        ckg[k0 / CB] = g;
        ckq[k0 / CB] = qp;
        double r[CB];
#pragma unroll
        for (int i = 0; i < CB; ++i) r[i] = (k0 + i < nz) ? col[(size_t)(k0 + i) * plane] : 0.0;
#pragma unroll
        for (int i = 0; i < CB; ++i) {
            const int k = k0 + i;
            if (k < nz) {
                const double bk = (k == 0) ? bfirst : ((k == nz - 1) ? blast : b);
                const double wk = (k == 0) ? gamma : ((k == nz - 1) ? 1.0 : 0.0);
                g = 1.0 / (bk - g);
                xp = (r[i] * scale - xp) * g;
                qp = (wk - qp) * g;
                if (!pin) col[(size_t)k * plane] = xp;
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
            double gg = ckg[k0 / CB], qq = ckq[k0 / CB];
#pragma unroll
            for (int i = 0; i < CB; ++i) r[i] = (k0 + i < nz - 1) ? col[(size_t)(k0 + i) * plane] : 0.0;
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
                        if (!pin) col[(size_t)k * plane] = x;
                    } else {
                        if (!pin) col[(size_t)k * plane] = r[i] - fac * q;   // r holds x_k
                    }
                }
            }
        }
        if (sweep == 0) fac = (x + xlast / gamma) / (1.0 + q + qlast / gamma);
    }
    if (pin) zero_mode_line(col, plane, nz, p.bcz, scale, p.zero_scratch);
}

}  // namespace pp
