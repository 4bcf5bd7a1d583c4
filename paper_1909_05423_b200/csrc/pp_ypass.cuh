// y-pass kernels: the transform along y (stride = one x row), forward and inverse, in place.
//
// On one GPU the paper's chunk exchange + data shuffle before the y transform (PAPER.md:386-403,
// Fig. 13) becomes an in-HBM tiled transpose: a CTA owns T adjacent double2 columns (T*16 bytes
// contiguous per row) for all ny rows of one z plane, pulls them into registers with coalesced
// row-segment loads, runs the shared-memory FFT core down each column, and writes the tile back.
//
// The x-pass left every row as nx/2 double2 elements.  A double2 column is either
//   * a complex column  -- x periodic, column >= 1: (Re, Im) of one kx mode.  With y periodic it
//     gets a plain complex FFT (eq. 6); or
//   * a pair of independent real columns (x Neumann/Dirichlet; or column 0 of periodic x, which
//     holds the real kx = 0 and kx = nx/2 modes; or any column when y is Neumann/Dirichlet, whose
//     real transforms act on Re and Im separately).  The pair rides one complex FFT and is
//     separated by Hermitian symmetry exactly as in the x-pass.
// Row layout after the forward pass:
//   y periodic, complex column:  row m = Z_m
//   y periodic, real pair:       "half-complex" rows: row 0 = (A_0, B_0), row N/2 = (A_N/2, B_N/2),
//                                row m = (Re A_m, Re B_m), row N-m = (Im A_m, Im B_m), 0 < m < N/2
//   y Neumann / Dirichlet:       row m = (Ya_m, Yb_m)  (DCT-II / DST-II coefficients, eq. 7 / 9)
// In every case the modified wavenumber of row m is Table 2's evaluated at m,
// because the periodic eigenvalue is even in m -- so the z solve needs one table per axis.
#pragma once
#include <type_traits>

#include "pp_xpass.cuh"

namespace pp {

template <int T>
struct LayoutCol {
    int c;
    __device__ __forceinline__ int operator()(int i) const { return pad8(i) * T + c; }
};

// Tiles of 4 columns (N > 512): a quarter-warp -- the unit a 16-byte shared-memory access is served
// in -- is 4 columns x 2 consecutive rows (t even, t + 1), so the two rows must land in different halves
// of a 128-byte bank row.  The padded layout does that for the row patterns of radix-8 stages only; the
// leading radix-2 / radix-4 stage of the 1024- and 2048-point transforms stores rows that differ by
// R0 = 2^S and conflicts two-way.  Here the low bit of the row is XORed with bit S instead: rows i, i+1
// (i even: every load, every later store) and rows i, i + R0 (the first stage's stores) then always differ
// in that bit.  No padding needed.
template <int S>
struct LayoutColXor4 {
    int c;
    __device__ __forceinline__ int operator()(int i) const { return ((i ^ ((i >> S) & 1)) << 2) + c; }
};
template <int N, int T>
struct YLayout {
    static constexpr bool XOR4 = (T == 4) && ((N & (N - 1)) == 0) && (FftCfg<N>::R0 == 2 || FftCfg<N>::R0 == 4);
    using type = typename std::conditional<XOR4, LayoutColXor4<FftCfg<N>::R0 == 2 ? 1 : 2>, LayoutCol<T>>::type;
};

struct SyncCta {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};

#ifndef PP_Y_T
#define PP_Y_T 8          // double2 columns per CTA for N <= 512 (128-byte row segments)
#endif
#ifndef PP_Y_MINB
#define PP_Y_MINB 2       // __launch_bounds__ min CTAs per SM (caps registers) for CTAs of <= 512 threads
#endif

template <int N>
struct YCfg {
    static constexpr int P = FftCfg<N>::P;
    static constexpr int T = (N <= 512) ? PP_Y_T : 4;   // double2 columns per CTA
    static constexpr int THREADS = T * P;
    static constexpr int MINB = (THREADS <= 512) ? PP_Y_MINB : 1;
    static constexpr size_t SMEM = size_t(T) * FftCfg<N>::SMEM_ELEMS * sizeof(double2);
};

__device__ __forceinline__ double2 dscale(double a, double2 v) { return make_double2(a * v.x, a * v.y); }

template <bool LDCG>
__device__ __forceinline__ double2 yld(const double2 *p) { return LDCG ? __ldcg(p) : *p; }

// One CTA-wide tile of the forward y pass: column tile bx (T double2 columns) of plane z, all N rows
// (blockDim.x == T * FftCfg<N>::P).  `smem` holds T * FftCfg<N>::SMEM_ELEMS double2.  LDCG: read with
// ld.global.cg -- for the fused x+y kernel, whose input was just written by other SMs.
template <int N, bool LDCG>
__device__ __forceinline__ void yfwd_tile(double2 *w, int nxh, int bc, int complex_cols,
                                          const double2 *__restrict__ tw, const double2 *__restrict__ ptw,
                                          int bx, int z, double2 *smem) {
    using C = FftCfg<N>;
    constexpr int E = C::E, P = C::P, T = YCfg<N>::T, H = N / 2;
    const int c = threadIdx.x % T, t = threadIdx.x / T;
    const int cp = bx * T + c;
    const bool active = cp < nxh;
    double2 *base = w + (size_t)z * N * nxh + (active ? cp : 0);
    const int ld = nxh;                                    // row offsets inside a plane fit 32 bits
    const typename YLayout<N, T>::type lay{c};
    const SyncCta sync;

    double2 v[E];
#pragma unroll
    for (int q = 0; q < E; ++q) {
        const int i = t + q * P;
        if (bc == BC_P) {
            v[q] = yld<LDCG>(base + i * ld);
        } else if (bc == BC_N) {
            const int p = (i < H) ? 2 * i : 2 * (N - 1 - i) + 1;
            v[q] = yld<LDCG>(base + p * ld);
        } else {
            if (i < H) v[q] = yld<LDCG>(base + (N - 1 - 2 * i) * ld);
            else       v[q] = dscale(-1.0, yld<LDCG>(base + (2 * i - N) * ld));
        }
    }

    fft<N, FWD>(v, t, smem, tw, lay, sync);

    if (complex_cols && bx > 0) {                  // block-uniform: all columns complex
        if (active) {
#pragma unroll
            for (int q = 0; q < E; ++q) base[(t + q * P) * ld] = v[q];
        }
        return;
    }
#pragma unroll
    for (int q = E / 2; q < E; ++q) smem[lay(t + q * P)] = v[q];       // partners live in the upper half
    __syncthreads();
    if (!active) return;
    if (complex_cols && cp > 0) {
#pragma unroll
        for (int q = 0; q < E; ++q) base[(t + q * P) * ld] = v[q];
        return;
    }
#pragma unroll
    for (int q = 0; q < E / 2; ++q) {
        const int m = t + q * P;
        const double2 zm = v[q];
        const double2 zc = smem[lay(neg_mod<N>(m))];
        if (m == 0) {
            const double2 zh = v[E / 2];
            if (bc == BC_P) {
                base[0] = zm;
                base[H * ld] = zh;
            } else {
                const double c4 = ptw[H].x;
                if (bc == BC_N) {
                    base[0] = zm;
                    base[H * ld] = dscale(c4, zh);
                } else {
                    base[(N - 1) * ld] = dscale(-1.0, zm);
                    base[(N - 1 - H) * ld] = dscale(-sgn_of(H) * c4, zh);
                }
            }
        } else {
            const double2 A = make_double2(0.5 * (zm.x + zc.x), 0.5 * (zm.y - zc.y));
            const double2 B = make_double2(0.5 * (zm.y + zc.y), -0.5 * (zm.x - zc.x));
            if (bc == BC_P) {
                base[m * ld] = make_double2(A.x, B.x);
                base[(N - m) * ld] = make_double2(A.y, B.y);
            } else {
                const double2 wm = __ldg(&ptw[m]);
                const double2 ca = cmul(wm, A), cb = cmul(wm, B);
                if (bc == BC_N) {
                    base[m * ld] = make_double2(ca.x, cb.x);
                    base[(N - m) * ld] = make_double2(-ca.y, -cb.y);
                } else {
                    const double s1 = -sgn_of(m);
                    base[(N - 1 - m) * ld] = make_double2(s1 * ca.x, s1 * cb.x);
                    base[(m - 1) * ld] = make_double2(-s1 * ca.y, -s1 * cb.y);
                }
            }
        }
    }
}


template <int N>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
ypass_fwd_kernel(double2 *w, int nxh, int bc, int complex_cols,
                 const double2 *__restrict__ tw, const double2 *__restrict__ ptw) {
    extern __shared__ double2 smem[];
    // planes from the last to the first: the x pass before this one went first to last, so the planes
    // it wrote last are still (dirty) in L2 -- they are read from there and overwritten there
    yfwd_tile<N, false>(w, nxh, bc, complex_cols, tw, ptw, blockIdx.x, gridDim.y - 1 - blockIdx.y, smem);
}

// One CTA-wide tile of the inverse y pass (see yfwd_tile).
template <int N>
__device__ __forceinline__ void yinv_tile(double2 *w, int nxh, int bc, int complex_cols,
                                          const double2 *__restrict__ tw, const double2 *__restrict__ ptw,
                                          int bx, int z, double2 *smem) {
    using C = FftCfg<N>;
    constexpr int E = C::E, P = C::P, T = YCfg<N>::T, H = N / 2;
    const int c = threadIdx.x % T, t = threadIdx.x / T;
    const int cp = bx * T + c;
    const bool active = cp < nxh;
    double2 *base = w + (size_t)z * N * nxh + (active ? cp : 0);
    const int ld = nxh;                                    // row offsets inside a plane fit 32 bits
    const typename YLayout<N, T>::type lay{c};
    const SyncCta sync;
    const bool cplx = complex_cols && cp > 0;

    double2 v[E];
    if (complex_cols && bx > 0) {                          // block-uniform: every column of the tile is complex
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = base[(t + q * P) * ld];
    } else {
        // Real pairs: row m and row N-m are needed together, for V_m and for V_{N-m}.  The owner of
        // m in [0, N/2) loads the two rows once, keeps V_m and hands V_{N-m} to its owner through shared
        // memory (thread 0 also makes V_{N/2}).  A complex column inside such a tile (periodic x and y,
        // first tile) just loads its eight rows and takes part in the barriers.
        // All loads first, so that they are in flight together; then the arithmetic.
        // (the upper half of v is the landing place of the second row of each pair)
        double2 yh = make_double2(0.0, 0.0);
#pragma unroll
        for (int q = 0; q < E / 2; ++q) {
            const int m = t + q * P;                       // 0 <= m < N/2
            if (cplx) {
                v[q] = base[m * ld];
                v[q + E / 2] = base[(m + H) * ld];
            } else if (bc == BC_P || bc == BC_N) {
                v[q] = base[m * ld];
                v[q + E / 2] = (m > 0) ? base[(N - m) * ld] : make_double2(0.0, 0.0);
                if (m == 0) yh = base[H * ld];
            } else {
                v[q] = base[(N - 1 - m) * ld];
                v[q + E / 2] = (m > 0) ? base[(m - 1) * ld] : make_double2(0.0, 0.0);
                if (m == 0) yh = base[(N - 1 - H) * ld];
            }
        }
        if (!cplx) {
#pragma unroll
            for (int q = 0; q < E / 2; ++q) {
                const int m = t + q * P;
                if (bc == BC_P) {
                    if (m == 0) {                          // (A, B) both real: Z = A + i B
                        smem[lay(H)] = yh;
                    } else {
                        const double2 lo = v[q], hi = v[q + E / 2];
                        v[q] = make_double2(lo.x - hi.y, hi.x + lo.y);
                        smem[lay(N - m)] = make_double2(lo.x + hi.y, lo.y - hi.x);
                    }
                } else {
                    const double s1 = (bc == BC_N) ? 1.0 : sgn_of(m);  // Dirichlet: Y'_m = (-1)^m S_{N-1-m}
                    const double2 a = dscale(s1, v[q]), b = dscale(s1, v[q + E / 2]);
                    const double2 wm = __ldg(&ptw[m]);
                    v[q] = cmul(cconj(wm), make_double2(a.x + b.y, a.y - b.x));
                    if (m > 0) {                           // conj(w_{N-m}) = i w_m
                        smem[lay(N - m)] = cmul(make_double2(-wm.y, wm.x), make_double2(b.x + a.y, b.y - a.x));
                    } else {
                        const double2 h2 = dscale((bc == BC_N) ? 1.0 : sgn_of(H), yh);
                        smem[lay(H)] = cmul(cconj(__ldg(&ptw[H])), make_double2(h2.x + h2.y, h2.y - h2.x));
                    }
                }
            }
        }
        sync();
        if (!cplx) {
#pragma unroll
            for (int q = E / 2; q < E; ++q) v[q] = smem[lay(t + q * P)];
        }
        sync();
    }
    // in place: every load of the tile precedes every store -- the barriers above and the FFT's
    // exchanges are CTA-wide; a single-stage transform has P = 1 (one thread owns the whole column)

    fft<N, INV>(v, t, smem, tw, lay, sync);

    if (!active) return;
#pragma unroll
    for (int q = 0; q < E; ++q) {
        const int i = t + q * P;
        if (bc == BC_P) {
            base[i * ld] = v[q];
        } else {
            const int p = (i < H) ? 2 * i : 2 * (N - 1 - i) + 1;
            if (bc == BC_N) base[p * ld] = v[q];
            else            base[(N - 1 - p) * ld] = dscale(-sgn_of(p), v[q]);
        }
    }
}


template <int N>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
ypass_inv_kernel(double2 *w, int nxh, int bc, int complex_cols,
                 const double2 *__restrict__ tw, const double2 *__restrict__ ptw) {
    extern __shared__ double2 smem[];
    yinv_tile<N>(w, nxh, bc, complex_cols, tw, ptw, blockIdx.x, blockIdx.y, smem);
}

}  // namespace pp
