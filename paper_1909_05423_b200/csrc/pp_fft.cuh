// Complex FFT core shared by the x- and y-pass kernels: a register + shared-memory Stockham
// autosort FFT, fp64.  Powers of two: radix 8 (leading radix 2 or 4 when log2 N is not a multiple
// of 3), or -- long transforms, 16 elements per thread -- radix 16 (leading radix 2, 4 or 8): one
// shared-memory exchange fewer at N = 1024 and 2048, where the exchanges are what the pass costs.
// 3 * 2^k and 5 * 2^k: a leading prime-factor butterfly of 6 / 12 / 10 / 20 points, then radix 4.
//
// "PittPack performs complex FFT transform for all the transformations": every
// periodic / Neumann / Dirichlet transform of the solver is this core plus a fused pre- and
// post-processing step.  The paper calls cuFFT here; this is the hand-written
// replacement.
//
// Thread mapping.  An N-point transform is done by P = N/E threads, E elements per thread (8 or 16 for
// powers of two, 12 or 20 otherwise).  Thread t holds, before and after every stage and on exit, the
// elements with index t + m*P (m = 0..E-1) in natural order -- so global loads and stores of
// consecutive threads are contiguous, and the last stage needs no shared-memory round trip.  A stage
// of radix R does E/R butterflies per thread.  Between stages the data is exchanged through shared
// memory (one store + one load of each element), padded by one element every eight so that every
// 16-byte access pattern of the power-of-two schedule is bank-conflict free.
#pragma once
#include <cuda_runtime.h>

namespace pp {

constexpr int FWD = -1;   // exp(-2 pi i k n / N)   (eq. 6)
constexpr int INV = +1;   // exp(+2 pi i k n / N), unnormalised

__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n >> 1); }

// Supported lengths: N = odd * 2^k with odd in {1, 3, 5} -- the powers of two of BASELINE.json's grids
// and the 48- and 80-multiples of the paper's weak-scaling runs.
//   odd = 1: E = 8 elements per thread, radix-8 stages after a first stage of radix 2, 4 or 8; or
//            E = 16, radix-16 stages after a first stage of radix 2, 4, 8 or 16 (chosen per pass: fft_E)
//   odd = 3: E = 12, radix-4 stages after a first stage of radix 12 (k even) or 6 (k odd)
//   odd = 5: E = 20, radix-4 stages after a first stage of radix 20 (k even) or 10 (k odd)
// The first stage has no twiddles; its composite butterflies (6, 10, 12, 20) are prime-factor
// (Good-Thomas) combinations of a 3- or 5-point and a 2- or 4-point DFT, so they need none inside either.
// Every helper below takes the length n and the elements per thread e of the schedule.
__host__ __device__ constexpr int fft_odd_part(int n) { return (n % 2 == 0) ? fft_odd_part(n / 2) : n; }
__host__ __device__ constexpr int fft_log2_part(int n) { return ilog2(n / fft_odd_part(n)); }
__host__ __device__ constexpr bool fft_length_ok(int n) {
    return n >= 4 && (fft_odd_part(n) == 1 || ((fft_odd_part(n) == 3 || fft_odd_part(n) == 5) && fft_log2_part(n) >= 4));
}
// elements per thread: powers of two from `e16_min` on take 16, shorter ones 8
__host__ __device__ constexpr int fft_E(int n, int e16_min) {
    return fft_odd_part(n) == 1 ? ((n >= e16_min && n >= 32) ? 16 : (n >= 8 ? 8 : n)) : 4 * fft_odd_part(n);
}
__host__ __device__ constexpr int stage_radix(int n, int e) { return fft_odd_part(n) == 1 ? (e == 16 ? 16 : 8) : 4; }   // every stage after the first
__host__ __device__ constexpr int first_radix(int n, int e) {
    return fft_odd_part(n) != 1 ? fft_odd_part(n) * ((fft_log2_part(n) % 2 == 0) ? 4 : 2)
         : e == 16 ? ((ilog2(n) % 4 == 0) ? 16 : (1 << (ilog2(n) % 4)))
                   : ((ilog2(n) % 3 == 0) ? 8 : ((ilog2(n) % 3 == 1) ? 2 : 4));
}

#ifndef PP_E16_MIN
#define PP_E16_MIN 1024       // default schedule: 16 elements per thread from this length on
#endif

__host__ __device__ constexpr int smem_stride(int elems, int p) {
    int s = elems;
    while ((s * 16) % 128 != (16 * p) % 128) ++s;
    return s;
}

template <int N, int E_ = fft_E(N, PP_E16_MIN)>
struct FftCfg {
    static_assert(fft_length_ok(N), "N = 2^k >= 4, or 3 * 2^k / 5 * 2^k with k >= 4");
    static constexpr int ODD = fft_odd_part(N);
    static constexpr int E = E_;                   // elements per thread
    static constexpr int P = N / E;                // threads per transform
    static constexpr int RS = stage_radix(N, E);   // radix of every stage after the first
    static constexpr int R0 = first_radix(N, E);   // first radix
    static constexpr int SMEM_ELEMS = N + N / 8;   // double2 elements per transform incl. padding
    // x pass, several transforms per CTA: distance between their scratch areas.  With P < 8 threads per transform a
    // quarter-warp spans 8 / P transforms, each touching P consecutive 16-byte slots: the areas are spaced so that those
    // runs tile one 128-byte bank row (stride = 16 P bytes modulo 128) instead of overlapping (ncu: half of the
    // 48-point x pass's shared-memory wavefronts were bank conflicts)
    static constexpr int SMEM_STRIDE = smem_stride(N + N / 8, P);
};

// Stage twiddle tables.  Every stage after the first has radix RS (16, 8 or 4) and multiplies input r of
// butterfly j by W_N^(k r STRIDE), k = j mod NS, STRIDE = N / (RS NS).  The plan stores, per stage, the
// row r = 1 (RS = 8, 16) or the rows r = 1, 2 (RS = 4) as [r][k] -- contiguous in k, so a warp's 16-byte loads
// touch NS*16 contiguous bytes instead of lines STRIDE*16 bytes apart; the other powers are products.
__host__ __device__ constexpr int tw_rows(int n, int e) { return stage_radix(n, e) == 4 ? 2 : 1; }
__host__ __device__ constexpr int tw_stage_offset(int n, int e, int NS) {
    int off = 0;
    for (int ns = first_radix(n, e); ns < NS; ns *= stage_radix(n, e)) off += tw_rows(n, e) * ns;
    return off;
}
__host__ __device__ constexpr int tw_table_elems(int n, int e) { return tw_stage_offset(n, e, n) > 0 ? tw_stage_offset(n, e, n) : 1; }

// (N - m) mod N for 0 <= m < N
template <int N>
__device__ __forceinline__ int neg_mod(int m) {
    if constexpr ((N & (N - 1)) == 0) return (N - m) & (N - 1);
    else return m == 0 ? 0 : N - m;
}

__device__ __forceinline__ int pad8(int i) { return i + (i >> 3); }

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 cconj(double2 a) { return make_double2(a.x, -a.y); }
// x or -x by the sign bit of the high word: the (-1)^m factors of the sine transform cost an integer
// instruction instead of a multiplication on the fp64 pipe; bit-identical to x * (+-1.0)
__device__ __forceinline__ double neg_if(double x, bool neg) {
    return __hiloint2double(__double2hiint(x) ^ (neg ? (int)0x80000000 : 0), __double2loint(x));
}
__device__ __forceinline__ double2 neg_if(double2 a, bool neg) { return make_double2(neg_if(a.x, neg), neg_if(a.y, neg)); }

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

// multiply by the constant (cr + i DIR ci): the forward twiddle (cr, -ci) or its conjugate
template <int DIR>
__device__ __forceinline__ double2 cmul_const(double2 a, double cr, double ci) {
    const double si = (DIR == FWD) ? -ci : ci;
    return make_double2(fma(a.x, cr, -(a.y * si)), fma(a.x, si, a.y * cr));
}

// Post-/pre-twiddles of the cosine and sine transforms, w_m = exp(-i pi m / (2N)): thread t needs
// them at m = t + q P, q = 0 .. E/2 - 1, and w_{t + q P} = w_t exp(-i pi q / (2E)) -- one table load per thread, the
// other E/2 - 1 by a rotation through a compile-time constant (a table load issued between a tile's stores queues
// behind them: ncu showed one long-scoreboard wait per coefficient pair).  cos / sin of pi q / (2E) <= pi/4 by
// their Taylor series, evaluated at compile time.
__host__ __device__ constexpr double ct_cos(double x) {
    double sum = 1.0, term = 1.0;
    for (int k = 1; k <= 12; ++k) { term *= -x * x / double((2 * k - 1) * (2 * k)); sum += term; }
    return sum;
}
__host__ __device__ constexpr double ct_sin(double x) {
    double sum = x, term = x;
    for (int k = 1; k <= 12; ++k) { term *= -x * x / double((2 * k) * (2 * k + 1)); sum += term; }
    return sum;
}
template <int E>
struct PtwSteps {
    double c[E / 2 > 0 ? E / 2 : 1], s[E / 2 > 0 ? E / 2 : 1];
    constexpr PtwSteps() : c(), s() {
        for (int q = 0; q < E / 2; ++q) {
            c[q] = ct_cos(3.14159265358979323846 * q / (2.0 * E));
            s[q] = ct_sin(3.14159265358979323846 * q / (2.0 * E));
        }
    }
};
// w_{t + q P} from w_t (q a compile-time constant after unrolling)
#ifndef PP_PTW_ROT
#define PP_PTW_ROT 1
#endif
#ifndef PP_HOIST_ZC_MIN_E
#define PP_HOIST_ZC_MIN_E 16     // partner reads hoisted above the stores only where registers allow (16+ elements per thread: 128-register kernels)
#endif
template <int E>
__device__ __forceinline__ double2 ptw_rot(double2 w0, int q, const double2 *ptw = nullptr, int m = 0) {
    constexpr PtwSteps<E> st;
#if !PP_PTW_ROT
    return __ldg(&ptw[m]);
#endif
    if (q == 0) return w0;
    const double c = st.c[q], sn = -st.s[q];         // exp(-i a) = cos a - i sin a
    return make_double2(fma(w0.x, c, -(w0.y * sn)), fma(w0.x, sn, w0.y * c));
}

// in-place 16-point DFT, 16 = 4 x 4: 4-point DFTs over n1 (n = 4 n1 + n0), twiddles W_16^(n0 k1), 4-point DFTs
// over n0.  The result is left transposed: X_{k1 + 4 k2} sits in x[4 k1 + k2] -- read it through bfly16_at.
__host__ __device__ constexpr int bfly16_at(int k) { return 4 * (k & 3) + (k >> 2); }
template <int DIR>
__device__ __forceinline__ void bfly16(double2 (&x)[16]) {
    constexpr double C = 0.92387953251128675613, S = 0.38268343236508977173, H = 0.70710678118654752440;
#pragma unroll
    for (int n0 = 0; n0 < 4; ++n0) bfly4<DIR>(x[n0], x[n0 + 4], x[n0 + 8], x[n0 + 12]);   // -> x[n0 + 4 k1]
    // W_16^(n0 k1) = cos(2 pi m / 16) + i DIR sin(2 pi m / 16), m = n0 k1 in {1, 2, 3, 2, 4, 6, 3, 6, 9}
    x[1 + 4] = cmul_const<DIR>(x[1 + 4], C, S);
    x[2 + 4] = cmul_const<DIR>(x[2 + 4], H, H);
    x[3 + 4] = cmul_const<DIR>(x[3 + 4], S, C);
    x[1 + 8] = cmul_const<DIR>(x[1 + 8], H, H);
    x[2 + 8] = rot90<DIR>(x[2 + 8]);
    x[3 + 8] = cmul_const<DIR>(x[3 + 8], -H, H);
    x[1 + 12] = cmul_const<DIR>(x[1 + 12], S, C);
    x[2 + 12] = cmul_const<DIR>(x[2 + 12], -H, H);
    x[3 + 12] = cmul_const<DIR>(x[3 + 12], -C, -S);
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) bfly4<DIR>(x[4 * k1], x[4 * k1 + 1], x[4 * k1 + 2], x[4 * k1 + 3]);   // -> x[4 k1 + k2]
}

// in-place natural-order 3-point DFT
template <int DIR>
__device__ __forceinline__ void bfly3(double2 &x0, double2 &x1, double2 &x2) {
    constexpr double S = 0.86602540378443864676;   // sin(2 pi / 3)
    const double2 t = cadd(x1, x2), u = csub(x1, x2);
    const double2 m = make_double2(fma(-0.5, t.x, x0.x), fma(-0.5, t.y, x0.y));
    // forward: x1' = m - i S u, x2' = m + i S u;  inverse: the other way round
    const double2 r = DIR == FWD ? make_double2(S * u.y, -S * u.x) : make_double2(-S * u.y, S * u.x);
    x0 = cadd(x0, t);
    x1 = cadd(m, r);
    x2 = csub(m, r);
}

// in-place natural-order 5-point DFT
template <int DIR>
__device__ __forceinline__ void bfly5(double2 &x0, double2 &x1, double2 &x2, double2 &x3, double2 &x4) {
    constexpr double C1 = 0.30901699437494742410, C2 = -0.80901699437494742410;   // cos(2 pi/5), cos(4 pi/5)
    constexpr double S1 = 0.95105651629515357212, S2 = 0.58778525229247312917;    // sin(2 pi/5), sin(4 pi/5)
    const double2 a = cadd(x1, x4), b = csub(x1, x4), c = cadd(x2, x3), d = csub(x2, x3);
    const double2 m1 = make_double2(x0.x + C1 * a.x + C2 * c.x, x0.y + C1 * a.y + C2 * c.y);
    const double2 m2 = make_double2(x0.x + C2 * a.x + C1 * c.x, x0.y + C2 * a.y + C1 * c.y);
    const double2 n1 = make_double2(S1 * b.x + S2 * d.x, S1 * b.y + S2 * d.y);
    const double2 n2 = make_double2(S2 * b.x - S1 * d.x, S2 * b.y - S1 * d.y);
    // forward: X_k = m -/+ i n  (k = 1, 2 take "- i n"), inverse: conjugate pattern
    const double2 r1 = DIR == FWD ? make_double2(n1.y, -n1.x) : make_double2(-n1.y, n1.x);
    const double2 r2 = DIR == FWD ? make_double2(n2.y, -n2.x) : make_double2(-n2.y, n2.x);
    x0 = cadd(x0, cadd(a, c));
    x1 = cadd(m1, r1);
    x4 = csub(m1, r1);
    x2 = cadd(m2, r2);
    x3 = csub(m2, r2);
}

// in-place natural-order DFT of length R = A * B, A in {3, 5}, B in {2, 4}: prime-factor (Good-Thomas)
// algorithm.  With input n = (B n1 + A n2) mod R and output k = (B b' k1 + A a' k2) mod R, where
// b' = B^-1 mod A and a' = A^-1 mod B, the kernel factors exactly into W_A^(n1 k1) W_B^(n2 k2): A-point
// DFTs over n1, then B-point DFTs over n2, no twiddles in between.  All index maps are compile-time.
__host__ __device__ constexpr int inv_mod(int a, int m) {
    for (int i = 1; i < m; ++i) if ((a * i) % m == 1) return i;
    return 1;
}
template <int A, int B, int DIR>
__device__ __forceinline__ void bfly_pfa(double2 (&x)[A * B]) {
    constexpr int R = A * B;
    double2 y[A][B];
#pragma unroll
    for (int n2 = 0; n2 < B; ++n2) {
        double2 c[A];
#pragma unroll
        for (int n1 = 0; n1 < A; ++n1) c[n1] = x[(B * n1 + A * n2) % R];
        if constexpr (A == 3) bfly3<DIR>(c[0], c[1], c[2]);
        else bfly5<DIR>(c[0], c[1], c[2], c[3], c[4]);
#pragma unroll
        for (int k1 = 0; k1 < A; ++k1) y[k1][n2] = c[k1];
    }
    constexpr int CB = B * inv_mod(B % A, A), CA = A * inv_mod(A % B, B);
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) {
        if constexpr (B == 2) bfly2<DIR>(y[k1][0], y[k1][1]);
        else bfly4<DIR>(y[k1][0], y[k1][1], y[k1][2], y[k1][3]);
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) x[(CB * k1 + CA * k2) % R] = y[k1][k2];
    }
}

// where output r of bfly<R> is found
template <int R>
__host__ __device__ constexpr int bfly_at(int r) { return R == 16 ? bfly16_at(r) : r; }

template <int R, int DIR>
__device__ __forceinline__ void bfly(double2 (&x)[R]) {
    if constexpr (R == 2) bfly2<DIR>(x[0], x[1]);
    else if constexpr (R == 4) bfly4<DIR>(x[0], x[1], x[2], x[3]);
    else if constexpr (R == 8) bfly8<DIR>(x);
    else if constexpr (R == 16) bfly16<DIR>(x);
    else if constexpr (R == 6) bfly_pfa<3, 2, DIR>(x);
    else if constexpr (R == 12) bfly_pfa<3, 4, DIR>(x);
    else if constexpr (R == 10) bfly_pfa<5, 2, DIR>(x);
    else bfly_pfa<5, 4, DIR>(x);
}

// One Stockham stage of radix R with NS = product of the previous radices.
//   butterfly j (0 <= j < N/R), k = j mod NS:
//     inputs  data[j + r N/R] * W_N^(k r N/(NS R)),  r = 0..R-1
//     outputs out[(j / NS) NS R + k + q NS],          q = 0..R-1
// Thread t does the E/R butterflies j = t + b P; their inputs are exactly its elements t + m P.
template <int N, int E, int R, int NS, int DIR, class Layout, class Sync>
__device__ __forceinline__ void fft_stage(double2 (&v)[E], int t, double2 *s,
                                          const double2 *__restrict__ tw, const Layout &lay, const Sync &sync) {
    using C = FftCfg<N, E>;
    constexpr int P = C::P, B = E / R;
    constexpr bool LAST = (NS * R == N);
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const int j = t + b * P;
        double2 x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = v[b + B * r];
        const int k = j % NS;
        if constexpr (NS > 1 && R == 16) {
            // W^(k r STRIDE), r = 1..15, from the table's r = 1 by products (depth 4: relative error ~ 1e-15);
            // every power is used as soon as it exists, so few of them are live at a time
            const double2 *ts = tw + tw_stage_offset(N, E, NS);
            double2 w1 = __ldg(&ts[k]);
            if (DIR == INV) w1 = cconj(w1);
            const double2 w2 = cmul(w1, w1), w4 = cmul(w2, w2), w8 = cmul(w4, w4);
            const double2 w3 = cmul(w1, w2);
            x[1] = cmul(x[1], w1);   x[2] = cmul(x[2], w2);   x[3] = cmul(x[3], w3);   x[4] = cmul(x[4], w4);
            x[8] = cmul(x[8], w8);
            x[9] = cmul(x[9], cmul(w8, w1));   x[10] = cmul(x[10], cmul(w8, w2));   x[11] = cmul(x[11], cmul(w8, w3));
            const double2 w12 = cmul(w8, w4);
            x[12] = cmul(x[12], w12);
            x[13] = cmul(x[13], cmul(w12, w1));   x[14] = cmul(x[14], cmul(w12, w2));   x[15] = cmul(x[15], cmul(w12, w3));
            x[5] = cmul(x[5], cmul(w4, w1));   x[6] = cmul(x[6], cmul(w4, w2));   x[7] = cmul(x[7], cmul(w4, w3));
        } else if constexpr (NS > 1 && R == 8) {
            // W^(k r STRIDE): r = 1 from the stage table, the other six powers by products (two squarings and
            // four multiplies: the loads cost more than the arithmetic here; relative error of W^7 ~ 1e-15)
            const double2 *ts = tw + tw_stage_offset(N, E, NS);
            double2 w1 = __ldg(&ts[k]);
            if (DIR == INV) w1 = cconj(w1);
            const double2 w2 = cmul(w1, w1);
            const double2 w4 = cmul(w2, w2);
            const double2 w3 = cmul(w1, w2);
            x[1] = cmul(x[1], w1);
            x[2] = cmul(x[2], w2);
            x[3] = cmul(x[3], w3);
            x[4] = cmul(x[4], w4);
            x[5] = cmul(x[5], cmul(w1, w4));
            x[6] = cmul(x[6], cmul(w2, w4));
            x[7] = cmul(x[7], cmul(w3, w4));
        } else if constexpr (NS > 1) {
            static_assert(R == 4, "stages after the first are radix 16 / 8 (powers of two) or radix 4 (3 * 2^k, 5 * 2^k)");
            const double2 *ts = tw + tw_stage_offset(N, E, NS);
            double2 w1 = __ldg(&ts[k]);
            double2 w2 = __ldg(&ts[NS + k]);
            if (DIR == INV) { w1 = cconj(w1); w2 = cconj(w2); }
            x[1] = cmul(x[1], w1);
            x[2] = cmul(x[2], w2);
            x[3] = cmul(x[3], cmul(w1, w2));
        }
        bfly<R, DIR>(x);
        if constexpr (LAST) {
#pragma unroll
            for (int r = 0; r < R; ++r) v[b + B * r] = x[bfly_at<R>(r)];
        } else {
            const int j0 = ((j - k) * R) + k;      // (j / NS) * NS * R + k
#pragma unroll
            for (int r = 0; r < R; ++r) s[lay(j0 + r * NS)] = x[bfly_at<R>(r)];
        }
    }
    if constexpr (!LAST) {
        sync();
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = s[lay(t + m * P)];
        sync();
    }
}

template <int N, int E, int NS, int DIR, class Layout, class Sync>
__device__ __forceinline__ void fft_stages(double2 (&v)[E], int t, double2 *s,
                                           const double2 *__restrict__ tw, const Layout &lay, const Sync &sync) {
    constexpr int R = (NS == 1) ? FftCfg<N, E>::R0 : FftCfg<N, E>::RS;
    fft_stage<N, E, R, NS, DIR>(v, t, s, tw, lay, sync);
    if constexpr (NS * R < N) fft_stages<N, E, NS * R, DIR>(v, t, s, tw, lay, sync);
}

// N-point complex DFT (sign DIR, unnormalised), E elements per thread (deduced from v).  On entry and exit
// thread t (0 <= t < P = N / E) holds elements t + m P in v[m].  `s` is the transform's shared-memory scratch
// addressed through `lay`; `sync` synchronises the P threads of this transform.  On exit the scratch is free
// for reuse (the last exchange ends with a sync).
template <int N, int DIR, int E, class Layout, class Sync>
__device__ __forceinline__ void fft(double2 (&v)[E], int t, double2 *s,
                                    const double2 *__restrict__ tw, const Layout &lay, const Sync &sync) {
    fft_stages<N, E, 1, DIR>(v, t, s, tw, lay, sync);
}

}  // namespace pp
