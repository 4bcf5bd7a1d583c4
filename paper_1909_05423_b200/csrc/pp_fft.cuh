// Complex FFT core shared by the x- and y-pass kernels: a register + shared-memory Stockham
// autosort FFT, radix 8 (leading radix 2 or 4 when log2 N is not a multiple of 3), fp64.
//
// "PittPack performs complex FFT transform for all the transformations": every
// periodic / Neumann / Dirichlet transform of the solver is this core plus a fused pre- and
// post-processing step.  The paper calls cuFFT here; this is the hand-written
// replacement.
//
// Thread mapping.  An N-point transform is done by P = N/E threads, E = min(8, N) elements per
// thread.  Thread t holds, before and after every stage and on exit, the elements with index
// t + m*P (m = 0..E-1) in natural order -- so global loads and stores of consecutive threads are
// contiguous, and the last stage needs no shared-memory round trip.  Between stages the data is
// exchanged through shared memory (one store + one load of each element), padded by one element
// every eight so that every 16-byte access pattern of the schedule is bank-conflict free.
#pragma once
#include <cuda_runtime.h>

namespace pp {

constexpr int FWD = -1;   // exp(-2 pi i k n / N)   (eq. 6)
constexpr int INV = +1;   // exp(+2 pi i k n / N), unnormalised

__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n >> 1); }

template <int N>
struct FftCfg {
    static_assert(N >= 4 && (N & (N - 1)) == 0, "power of two >= 4");
    static constexpr int LOG2 = ilog2(N);
    static constexpr int E = N >= 8 ? 8 : N;       // elements per thread
    static constexpr int P = N / E;                // threads per transform
    static constexpr int R0 = (LOG2 % 3 == 0) ? 8 : ((LOG2 % 3 == 1) ? 2 : 4);   // first radix
    static constexpr int SMEM_ELEMS = N + N / 8;   // double2 elements per transform incl. padding
};

// Stage twiddle tables.  Every stage after the first is radix 8 and multiplies input r of butterfly
// j by W_N^(k r STRIDE), k = j mod NS, STRIDE = N / (8 NS).  The plan stores, per stage, the three
// rows r = 1, 2, 4 as [r][k] -- contiguous in k, so a warp's 16-byte loads touch NS*16 contiguous
// bytes (one L1 line for NS = 8, four for NS >= 32) instead of lines STRIDE*16 bytes apart; the other
// powers are products.  Stage with NS starts at element 3 * (sum of the earlier stages' NS).
__host__ __device__ constexpr int first_radix(int n) {
    return (ilog2(n) % 3 == 0) ? 8 : ((ilog2(n) % 3 == 1) ? 2 : 4);
}
__host__ __device__ constexpr int tw_stage_offset(int n, int NS) {
    int off = 0;
    for (int ns = first_radix(n); ns < NS; ns *= 8) off += 3 * ns;
    return off;
}
__host__ __device__ constexpr int tw_table_elems(int n) { return tw_stage_offset(n, n) > 0 ? tw_stage_offset(n, n) : 1; }

__device__ __forceinline__ int pad8(int i) { return i + (i >> 3); }

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 cconj(double2 a) { return make_double2(a.x, -a.y); }

// multiply by W_4 = exp(DIR * i pi/2):  forward -i, inverse +i
template <int DIR>
__device__ __forceinline__ double2 rot90(double2 a) {
    return DIR == FWD ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x);
}

template <int DIR>
__device__ __forceinline__ void bfly2(double2 &a, double2 &b) {
    double2 t = csub(a, b);
    a = cadd(a, b);
    b = t;
}

// in-place natural-order 4-point DFT of (x0,x1,x2,x3)
template <int DIR>
__device__ __forceinline__ void bfly4(double2 &x0, double2 &x1, double2 &x2, double2 &x3) {
    double2 t0 = cadd(x0, x2), t1 = csub(x0, x2);
    double2 t2 = cadd(x1, x3), t3 = rot90<DIR>(csub(x1, x3));
    x0 = cadd(t0, t2);
    x2 = csub(t0, t2);
    x1 = cadd(t1, t3);
    x3 = csub(t1, t3);
}

// in-place natural-order 8-point DFT
template <int DIR>
__device__ __forceinline__ void bfly8(double2 (&x)[8]) {
    constexpr double H = 0.70710678118654752440;   // sqrt(1/2)
    bfly4<DIR>(x[0], x[2], x[4], x[6]);            // even part  -> E0..E3 in x0,x2,x4,x6
    bfly4<DIR>(x[1], x[3], x[5], x[7]);            // odd part   -> O0..O3 in x1,x3,x5,x7
    // O1 *= W8, O2 *= W8^2, O3 *= W8^3
    double2 o1 = x[3], o2 = rot90<DIR>(x[5]), o3 = x[7];
    if (DIR == FWD) {
        o1 = make_double2((o1.x + o1.y) * H, (o1.y - o1.x) * H);       // (1-i)/sqrt2
        o3 = make_double2((o3.y - o3.x) * H, -(o3.x + o3.y) * H);      // (-1-i)/sqrt2
    } else {
        o1 = make_double2((o1.x - o1.y) * H, (o1.x + o1.y) * H);       // (1+i)/sqrt2
        o3 = make_double2(-(o3.x + o3.y) * H, (o3.x - o3.y) * H);      // (-1+i)/sqrt2
    }
    double2 e0 = x[0], e1 = x[2], e2 = x[4], e3 = x[6], o0 = x[1];
    x[0] = cadd(e0, o0); x[4] = csub(e0, o0);
    x[1] = cadd(e1, o1); x[5] = csub(e1, o1);
    x[2] = cadd(e2, o2); x[6] = csub(e2, o2);
    x[3] = cadd(e3, o3); x[7] = csub(e3, o3);
}

template <int R, int DIR>
__device__ __forceinline__ void bfly(double2 (&x)[R]) {
    if constexpr (R == 2) bfly2<DIR>(x[0], x[1]);
    else if constexpr (R == 4) bfly4<DIR>(x[0], x[1], x[2], x[3]);
    else bfly8<DIR>(x);
}

// One Stockham stage of radix R with NS = product of the previous radices.
//   butterfly j (0 <= j < N/R), k = j mod NS:
//     inputs  data[j + r N/R] * W_N^(k r N/(NS R)),  r = 0..R-1
//     outputs out[(j / NS) NS R + k + q NS],          q = 0..R-1
// Thread t does the E/R butterflies j = t + b P; their inputs are exactly its elements t + m P.
template <int N, int R, int NS, int DIR, class Layout, class Sync>
__device__ __forceinline__ void fft_stage(double2 (&v)[FftCfg<N>::E], int t, double2 *s,
                                          const double2 *__restrict__ tw, const Layout &lay, const Sync &sync) {
    using C = FftCfg<N>;
    constexpr int E = C::E, P = C::P, B = E / R;
    constexpr bool LAST = (NS * R == N);
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const int j = t + b * P;
        double2 x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = v[b + B * r];
        const int k = j & (NS - 1);
        if constexpr (NS > 1) {
            static_assert(R == 8, "every stage after the first is radix 8");
            // W^(k r STRIDE): load r = 1, 2, 4 from the stage table, build the rest with one product each
            const double2 *ts = tw + tw_stage_offset(N, NS);
            double2 w1 = __ldg(&ts[k]);
            double2 w2 = __ldg(&ts[NS + k]);
            double2 w4 = __ldg(&ts[2 * NS + k]);
            if (DIR == INV) { w1 = cconj(w1); w2 = cconj(w2); w4 = cconj(w4); }
            const double2 w3 = cmul(w1, w2);
            x[1] = cmul(x[1], w1);
            x[2] = cmul(x[2], w2);
            x[3] = cmul(x[3], w3);
            x[4] = cmul(x[4], w4);
            x[5] = cmul(x[5], cmul(w1, w4));
            x[6] = cmul(x[6], cmul(w2, w4));
            x[7] = cmul(x[7], cmul(w3, w4));
        }
        bfly<R, DIR>(x);
        if constexpr (LAST) {
#pragma unroll
            for (int r = 0; r < R; ++r) v[b + B * r] = x[r];
        } else {
            const int j0 = ((j - k) * R) + k;      // (j / NS) * NS * R + k
#pragma unroll
            for (int r = 0; r < R; ++r) s[lay(j0 + r * NS)] = x[r];
        }
    }
    if constexpr (!LAST) {
        sync();
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = s[lay(t + m * P)];
        sync();
    }
}

template <int N, int NS, int DIR, class Layout, class Sync>
__device__ __forceinline__ void fft_stages(double2 (&v)[FftCfg<N>::E], int t, double2 *s,
                                           const double2 *__restrict__ tw, const Layout &lay, const Sync &sync) {
    constexpr int R = (NS == 1) ? FftCfg<N>::R0 : 8;
    fft_stage<N, R, NS, DIR>(v, t, s, tw, lay, sync);
    if constexpr (NS * R < N) fft_stages<N, NS * R, DIR>(v, t, s, tw, lay, sync);
}

// N-point complex DFT (sign DIR, unnormalised).  On entry and exit thread t (0 <= t < P) holds
// elements t + m P in v[m].  `s` is the transform's shared-memory scratch addressed through `lay`;
// `sync` synchronises the P threads of this transform.  On exit the scratch is free for reuse
// (the last exchange ends with a sync).
template <int N, int DIR, class Layout, class Sync>
__device__ __forceinline__ void fft(double2 (&v)[FftCfg<N>::E], int t, double2 *s,
                                    const double2 *__restrict__ tw, const Layout &lay, const Sync &sync) {
    fft_stages<N, 1, DIR>(v, t, s, tw, lay, sync);
}

}  // namespace pp
