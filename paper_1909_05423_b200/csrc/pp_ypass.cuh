// y-pass kernels: the transform along y (stride = one x row), forward and inverse, in place.
//
// On one GPU the paper's chunk exchange + data shuffle before the y transform (PAPER.md:386-403,
// Fig. 13) becomes an in-HBM tiled transpose: a CTA owns T adjacent double2 columns (T*16 bytes
// contiguous per row) for all ny rows of one z plane, pulls them into registers -- with coalesced
// row-segment loads (ny <= 512), or through TMA box copies into its shared-memory tile (ny >= 1024) --,
// runs the shared-memory FFT core down each column, and writes the tile back.
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

#include "pp_tma.cuh"
#include "pp_xpass.cuh"

namespace pp {

template <int T>
struct LayoutCol {
    int c;
    __device__ __forceinline__ int operator()(int i) const { return pad8(i) * T + c; }
};

// Tiles of fewer than 8 columns (N > 512).  A quarter-warp -- the unit a 16-byte shared-memory access is
// served in -- is T columns x 8/T consecutive rows (t aligned to 8/T), so those 8/T rows must land in
// different T*16-byte slices of a 128-byte bank row.  The padded layout does that for the row patterns of
// radix-8 stages on 8 columns only.  Here the low log2(8/T) bits of the row are XORed with the bits just
// above the first radix R0 = 2^S instead:
//   loads (rows t + m P) and the stores of every later stage (rows .. + k, k = t mod NS): the 8/T rows are
//     consecutive and share the XORed bits -- still distinct;
//   stores of the first stage (rows t R0 + r): the rows differ in exactly the bits S.. that are XORed in.
// No padding needed.
template <int T, int S>
struct LayoutColXor {
    static constexpr int MASK = 8 / T - 1;
    int c;
    __device__ __forceinline__ int operator()(int i) const { return (i ^ ((i >> S) & MASK)) * T + c; }
};

struct SyncCta {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};

#ifndef PP_Y_T
#define PP_Y_T 8          // double2 columns per CTA for N <= 512 (128-byte row segments)
#endif
#ifndef PP_Y_T_1024
#define PP_Y_T_1024 4     // ... for N in (512, 1024]
#endif
#ifndef PP_Y_T_2048
#define PP_Y_T_2048 2     // ... for N > 1024 (32-byte row segments: two resident CTAs per SM beat one with 64-byte ones, measured)
#endif
#ifndef PP_Y_MINB
#define PP_Y_MINB 2       // __launch_bounds__ min CTAs per SM (caps registers) for CTAs of <= 512 threads
#endif
#ifndef PP_Y_E16_MIN
#define PP_Y_E16_MIN 1024 // y pass: 16 elements per thread (radix-16 stages) from this length on
#endif

template <int N>
struct YCfg {
    static constexpr int E = fft_E(N, PP_Y_E16_MIN);
    using F = FftCfg<N, E>;
    static constexpr int P = F::P;
    static constexpr int T = (N <= 512) ? PP_Y_T : ((N <= 1024) ? PP_Y_T_1024 : PP_Y_T_2048);   // double2 columns per CTA
    static constexpr int THREADS = T * P;
    // registers: 8 elements per thread fit 64 (two CTAs of 512 threads per SM); 16 or 20 need up to 128
    static constexpr int MINB = (E <= 12) ? ((THREADS <= 512) ? PP_Y_MINB : 1) : ((THREADS <= 256) ? 2 : 1);
    static constexpr bool XOR = (T < 8) && ((N & (N - 1)) == 0) && (N > 512);
    using Layout = typename std::conditional<XOR, LayoutColXor<T, ilog2(F::R0)>, LayoutCol<T>>::type;
    static constexpr size_t SMEM = size_t(T) * (XOR ? N : F::SMEM_ELEMS) * sizeof(double2);
};

__device__ __forceinline__ double2 dscale(double a, double2 v) { return make_double2(a * v.x, a * v.y); }

template <bool LDCG>
__device__ __forceinline__ double2 yld(const double2 *p) { return LDCG ? __ldcg(p) : *p; }

// Slab decomposition over several GPUs (pp_slab_*): the y pass is where the data is
// re-oriented between z-slabs (x and y transforms local) and (kx, ky)-pencils (z solve local),
// so the exchange is fused into it -- the forward pass STORES row j of plane z straight into the pencil
// buffer of the rank that owns ky = j (a peer pointer over NVLink, or a chunk of a local all-to-all send
// buffer), the inverse pass LOADS it from there.  Block b = j / rpb of `rpb` consecutive rows lives at
// base[b], laid out [plane z][row j - b rpb][nxh]: with one block (rpb = ny) this is the plain array.
constexpr int PP_MAX_WORLD = 16;
struct YRows {
    double2 *base[PP_MAX_WORLD];
    int rpb;
    __device__ __forceinline__ double2 *row(int z, int j, int ld) const {
        const int b = j / rpb;
        return base[b] + ((size_t)z * rpb + (j - b * rpb)) * (size_t)ld;
    }
};

// ---- double-buffered staging with cp.async (persistent kernel; a build switch, off: measured slower -- the second
// buffer costs one of the two resident CTAs; the tiles that ARE staged go through TMA into the
// exchange buffer itself, see ypass_*_tma_kernel below) ---------------------------------------------------------
// A resident CTA walks over tiles and copies its NEXT tile from global into a second shared-memory buffer with
// asynchronous 16-byte copies (cp.async / LDGSTS: no registers, no scoreboard wait) while it transforms the current
// one -- the load latency that the plain kernels expose once per tile (ncu: long-scoreboard stalls, one or two
// resident CTAs per SM at N >= 1024) is hidden behind a whole tile of arithmetic.  The copy applies the pass's row
// permutation on the way, so the staged tile is read back in natural order: rows t, t+1 of
// a quarter-warp are adjacent, conflict-free without padding.
__device__ __forceinline__ void cp_async16(double2 *smem_dst, const double2 *gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

struct NoHook {
    __device__ __forceinline__ void operator()() const {}
};

#ifndef PP_Y_STAGED_MIN
#define PP_Y_STAGED_MIN 4096      // y pass: staged persistent kernel from this length on (4096: never)
#endif
template <int N>
struct YStaged {
    static constexpr bool ON = (N >= PP_Y_STAGED_MIN);
    static constexpr size_t IN_BYTES = size_t(YCfg<N>::T) * N * sizeof(double2);
    static constexpr size_t SMEM = YCfg<N>::SMEM + IN_BYTES;
    static constexpr int PER_SM_SMEM = int((227 * 1024) / (SMEM + 1024));
    static constexpr int PER_SM_THREADS = 2048 / YCfg<N>::THREADS;
    static constexpr int REGS = (YCfg<N>::E <= 12 && YCfg<N>::E != 12) ? 64 : 128;
    static constexpr int PER_SM_REGS = 65536 / (REGS * YCfg<N>::THREADS);
    static constexpr int PER_SM0 = PER_SM_SMEM < PER_SM_THREADS ? PER_SM_SMEM : PER_SM_THREADS;
    static constexpr int PER_SM = (PER_SM0 < PER_SM_REGS ? PER_SM0 : PER_SM_REGS) > 0 ? (PER_SM0 < PER_SM_REGS ? PER_SM0 : PER_SM_REGS) : 1;
};

// copies of one tile of the forward pass into `stage`: position i <- the row the transform wants at input i
template <int N>
__device__ __forceinline__ void yfwd_stage_issue(const double2 *w, int nxh, int bc, int bx, int z, double2 *stage) {
    using C = typename YCfg<N>::F;
    constexpr int E = C::E, P = C::P, T = YCfg<N>::T, H = N / 2;
    const int c = threadIdx.x % T, t = threadIdx.x / T;
    const int cp = bx * T + c;
    const double2 *base = w + (size_t)z * N * nxh + (cp < nxh ? cp : 0);
#pragma unroll
    for (int q = 0; q < E; ++q) {
        const int i = t + q * P;
        int row = i;
        if (bc == BC_N) row = (i < H) ? 2 * i : 2 * (N - 1 - i) + 1;
        else if (bc == BC_D) row = (i < H) ? N - 1 - 2 * i : 2 * i - N;
        cp_async16(stage + i * T + c, base + row * nxh);
    }
    cp_async_commit();
}
// ... of the inverse pass: rows in natural order
template <int N>
__device__ __forceinline__ void yinv_stage_issue(const double2 *w, int nxh, int bx, int z, double2 *stage) {
    using C = typename YCfg<N>::F;
    constexpr int E = C::E, P = C::P, T = YCfg<N>::T;
    const int c = threadIdx.x % T, t = threadIdx.x / T;
    const int cp = bx * T + c;
    const double2 *base = w + (size_t)z * N * nxh + (cp < nxh ? cp : 0);
#pragma unroll
    for (int q = 0; q < E; ++q) {
        const int j = t + q * P;
        cp_async16(stage + j * T + c, base + j * nxh);
    }
    cp_async_commit();
}

// One CTA-wide tile of the forward y pass: column tile bx (T double2 columns) of plane z, all N rows
// (blockDim.x == YCfg<N>::THREADS).  `smem` holds YCfg<N>::SMEM bytes.  LDCG: read with
// ld.global.cg -- for the fused x+y kernel, whose input was just written by other SMs.
// STAGED: the tile's input was copied to `stage` by yfwd_stage_issue; `after_load` runs when every thread has its
// input in registers (the staged kernel puts a barrier and the next tile's copies there).
// (STAGED: 0 no; 1 `stage` holds the permuted sequence, position i = input i (cp.async kernel); 2 `stage` holds the rows
// as the tensor maps of the TMA kernel deliver them: periodic: row i at i; Neumann / Dirichlet: even rows 0, 2, ... at
// 0 .. N/2-1, odd rows 1, 3, ... at N/2 .. N-1)
template <int N, bool LDCG, bool SLAB = false, int STAGED = 0, class Hook = NoHook>
__device__ __forceinline__ void yfwd_tile(double2 *w, int nxh, int bc, int complex_cols,
                                          const double2 *__restrict__ tw, const double2 *__restrict__ ptw,
                                          int bx, int z, double2 *smem, const YRows *rows = nullptr,
                                          const double2 *stage = nullptr, const Hook &after_load = Hook()) {
    using C = typename YCfg<N>::F;
    constexpr int E = C::E, P = C::P, T = YCfg<N>::T, H = N / 2;
    const int c = threadIdx.x % T, t = threadIdx.x / T;
    const int cp = bx * T + c;
    const bool active = cp < nxh;
    double2 *base = w + (size_t)z * N * nxh + (active ? cp : 0);
    const int ld = nxh;                                    // row offsets inside a plane fit 32 bits
    const typename YCfg<N>::Layout lay{c};
    const SyncCta sync;
    // where row j of the result goes: in place, or (slab decomposition) into the owner rank's pencil block
    const auto out = [&](int j) -> double2 * {
        if constexpr (SLAB) return rows->row(z, j, ld) + (active ? cp : 0);
        else return base + j * ld;
    };

    double2 v[E];
#pragma unroll
    for (int q = 0; q < E; ++q) {
        const int i = t + q * P;
        if constexpr (STAGED == 1) {
            v[q] = stage[i * T + c];
            if (bc == BC_D && i >= H) v[q] = dscale(-1.0, v[q]);
        } else if constexpr (STAGED == 2) {
            // v_i = row 2i (i < H), row 2(N-1-i)+1 otherwise (Neumann); row N-1-2i, -row(2i-N) (Dirichlet): every run of
            // consecutive i is a run of consecutive staged rows, ascending or descending (conflict-free either way)
            const int pos = (bc == BC_P) ? i : ((bc == BC_N) ? ((i < H) ? i : H + (N - 1 - i)) : ((i < H) ? H + (H - 1 - i) : i - H));
            v[q] = stage[pos * T + c];
            if (bc == BC_D && i >= H) v[q] = dscale(-1.0, v[q]);
        } else if (bc == BC_P) {
            v[q] = yld<LDCG>(base + i * ld);
        } else if (bc == BC_N) {
            const int p = (i < H) ? 2 * i : 2 * (N - 1 - i) + 1;
            v[q] = yld<LDCG>(base + p * ld);
        } else {
            if (i < H) v[q] = yld<LDCG>(base + (N - 1 - 2 * i) * ld);
            else       v[q] = dscale(-1.0, yld<LDCG>(base + (2 * i - N) * ld));
        }
    }
    after_load();

    fft<N, FWD>(v, t, smem, tw, lay, sync);

    if (complex_cols && bx > 0) {                  // block-uniform: all columns complex
        if (active) {
#pragma unroll
            for (int q = 0; q < E; ++q) *out((t + q * P)) = v[q];
        }
        return;
    }
#pragma unroll
    for (int q = E / 2; q < E; ++q) smem[lay(t + q * P)] = v[q];       // partners live in the upper half
    __syncthreads();
    if (!active) return;
    if (complex_cols && cp > 0) {
#pragma unroll
        for (int q = 0; q < E; ++q) *out((t + q * P)) = v[q];
        return;
    }
    // the partners first, all in flight together, and one post-twiddle per thread (ptw_rot): loads issued between
    // the stores below queue behind them
    double2 zcs[E / 2];
    const double2 w0 = (bc != BC_P) ? __ldg(&ptw[t]) : make_double2(1.0, 0.0);
#pragma unroll
    for (int q = 0; q < E / 2; ++q) if (E >= PP_HOIST_ZC_MIN_E) zcs[q] = smem[lay(neg_mod<N>(t + q * P))];
#pragma unroll
    for (int q = 0; q < E / 2; ++q) {
        const int m = t + q * P;
        const double2 zm = v[q];
        const double2 zc = (E >= PP_HOIST_ZC_MIN_E) ? zcs[q] : smem[lay(neg_mod<N>(m))];
        if (m == 0) {
            const double2 zh = v[E / 2];
            if (bc == BC_P) {
                *out(0) = zm;
                *out(H) = zh;
            } else {
                constexpr double c4 = 0.70710678118654752440;      // cos(pi/4) = Re w_{N/2}
                if (bc == BC_N) {
                    *out(0) = zm;
                    *out(H) = dscale(c4, zh);
                } else {
                    *out((N - 1)) = dscale(-1.0, zm);
                    *out((N - 1 - H)) = dscale(-sgn_of(H) * c4, zh);
                }
            }
        } else {
            const double2 A = make_double2(0.5 * (zm.x + zc.x), 0.5 * (zm.y - zc.y));
            const double2 B = make_double2(0.5 * (zm.y + zc.y), -0.5 * (zm.x - zc.x));
            if (bc == BC_P) {
                *out(m) = make_double2(A.x, B.x);
                *out((N - m)) = make_double2(A.y, B.y);
            } else {
                const double2 wm = ptw_rot<E>(w0, q, ptw, m);
                const double2 ca = cmul(wm, A), cb = cmul(wm, B);
                if (bc == BC_N) {
                    *out(m) = make_double2(ca.x, cb.x);
                    *out((N - m)) = make_double2(-ca.y, -cb.y);
                } else {
                    const bool odd = m & 1;                        // logical m -> row N-1-m, sign -(-1)^m; logical N-m -> row m-1
                    *out((N - 1 - m)) = make_double2(neg_if(ca.x, !odd), neg_if(cb.x, !odd));
                    *out((m - 1)) = make_double2(neg_if(ca.y, odd), neg_if(cb.y, odd));
                }
            }
        }
    }
}


// L2 prefetch of a later tile (plain kernels, N >= PP_Y_PREFETCH_MIN): CTAs are handed out in the order of their linear
// block index, so the tile PP_Y_PREFETCH indices ahead is loaded by a CTA that starts about PP_Y_PREFETCH / (resident
// CTAs) tile lifetimes from now; one prefetch per row segment brings it into L2 meanwhile, and that CTA's load phase
// (ncu: long-scoreboard stalls with two resident CTAs per SM) waits for L2 instead of HBM.
#ifndef PP_Y_PREFETCH
#define PP_Y_PREFETCH 296      // tiles ahead (0: off): one wave of resident CTAs (2 x 148)
#endif
#ifndef PP_Y_PREFETCH_MIN
#define PP_Y_PREFETCH_MIN 1024 // measured: +7 % at N = 1024 (64-byte row segments, load phase 30 % of a tile's life),
#endif
#ifndef PP_Y_PREFETCH_MAX
#define PP_Y_PREFETCH_MAX 1024 // -5 % at N = 2048 (32-byte segments: the prefetches cost L1 tag cycles the pass is short of)
#endif
template <int N>
__device__ __forceinline__ void y_prefetch_ahead(const double2 *w, int nxh, bool reversed) {
    if constexpr (PP_Y_PREFETCH > 0 && N >= PP_Y_PREFETCH_MIN && N <= PP_Y_PREFETCH_MAX) {
        using C = typename YCfg<N>::F;
        constexpr int E = C::E, P = C::P, T = YCfg<N>::T;
        const int c = threadIdx.x % T, t = threadIdx.x / T;
        if (c != 0) return;
        const long long L = (long long)blockIdx.x + (long long)gridDim.x * blockIdx.y + PP_Y_PREFETCH;
        if (L >= (long long)gridDim.x * gridDim.y) return;
        const int bx = (int)(L % gridDim.x), by = (int)(L / gridDim.x);
        const int z = reversed ? (int)gridDim.y - 1 - by : by;
        const int col = bx * T < nxh ? bx * T : nxh - 1;
        const double2 *base = w + (size_t)z * N * nxh + col;
#pragma unroll
        for (int q = 0; q < E; ++q)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(base + (t + q * P) * nxh));
    }
}

template <int N>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
ypass_fwd_kernel(double2 *w, int nxh, int bc, int complex_cols,
                 const double2 *__restrict__ tw, const double2 *__restrict__ ptw) {
    extern __shared__ double2 smem[];
    // planes from the last to the first: the x pass before this one went first to last, so the planes
    // it wrote last are still (dirty) in L2 -- they are read from there and overwritten there
    y_prefetch_ahead<N>(w, nxh, true);
    yfwd_tile<N, false>(w, nxh, bc, complex_cols, tw, ptw, blockIdx.x, gridDim.y - 1 - blockIdx.y, smem);
}

// slab decomposition: reads the local z-slab w, stores every row into the pencil block of the rank that owns it
template <int N>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
ypass_fwd_slab_kernel(double2 *w, int nxh, int bc, int complex_cols,
                      const double2 *__restrict__ tw, const double2 *__restrict__ ptw, const __grid_constant__ YRows rows) {
    extern __shared__ double2 smem[];
    yfwd_tile<N, false, true>(w, nxh, bc, complex_cols, tw, ptw, blockIdx.x, gridDim.y - 1 - blockIdx.y, smem, &rows);
}

// One CTA-wide tile of the inverse y pass (see yfwd_tile).
// TSTORE: the result is left in `smem` for a TMA store instead of being stored (rows in the order of the tensor maps:
// periodic: row i at i; Neumann / Dirichlet: even rows at 0 .. N/2-1, odd rows at N/2 .. N-1, see y_tma_flush)
template <int N, bool SLAB = false, int STAGED = 0, class Hook = NoHook, bool TSTORE = false>
__device__ __forceinline__ void yinv_tile(double2 *w, int nxh, int bc, int complex_cols,
                                          const double2 *__restrict__ tw, const double2 *__restrict__ ptw,
                                          int bx, int z, double2 *smem, const YRows *rows = nullptr,
                                          const double2 *stage = nullptr, const Hook &after_load = Hook()) {
    using C = typename YCfg<N>::F;
    constexpr int E = C::E, P = C::P, T = YCfg<N>::T, H = N / 2;
    const int c = threadIdx.x % T, t = threadIdx.x / T;
    const int cp = bx * T + c;
    const bool active = cp < nxh;
    double2 *base = w + (size_t)z * N * nxh + (active ? cp : 0);
    const int ld = nxh;                                    // row offsets inside a plane fit 32 bits
    const typename YCfg<N>::Layout lay{c};
    const SyncCta sync;
    const bool cplx = complex_cols && cp > 0;
    // where row j of the input comes from: in place, or (slab decomposition) the owner rank's pencil block
    const auto in = [&](int j) -> const double2 * {
        if constexpr (STAGED) return stage + j * T + c;
        else if constexpr (SLAB) return rows->row(z, j, ld) + (active ? cp : 0);
        else return base + j * ld;
    };

    double2 v[E];
    if (complex_cols && bx > 0) {                          // block-uniform: every column of the tile is complex
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = *in((t + q * P));
        after_load();
    } else {
        // Real pairs: row m and row N-m are needed together, for V_m and for V_{N-m}.  The owner of
        // m in [0, N/2) loads the two rows once, keeps V_m and hands V_{N-m} to its owner through shared
        // memory (thread 0 also makes V_{N/2}).  A complex column inside such a tile (periodic x and y,
        // first tile) just loads its eight rows and takes part in the barriers.
        // All loads first, so that they are in flight together; then the arithmetic.
        // (the upper half of v is the landing place of the second row of each pair)
        double2 yh = make_double2(0.0, 0.0);
        // one pre-twiddle per thread, fetched with the rows; the others by rotation (ptw_rot)
        const double2 w0 = (!cplx && bc != BC_P) ? __ldg(&ptw[t]) : make_double2(1.0, 0.0);
#pragma unroll
        for (int q = 0; q < E / 2; ++q) {
            const int m = t + q * P;                       // 0 <= m < N/2
            if (cplx) {
                v[q] = *in(m);
                v[q + E / 2] = *in((m + H));
            } else if (bc == BC_P || bc == BC_N) {
                v[q] = *in(m);
                v[q + E / 2] = (m > 0) ? *in((N - m)) : make_double2(0.0, 0.0);
                if (m == 0) yh = *in(H);
            } else {
                v[q] = *in((N - 1 - m));
                v[q + E / 2] = (m > 0) ? *in((m - 1)) : make_double2(0.0, 0.0);
                if (m == 0) yh = *in((N - 1 - H));
            }
        }
        after_load();
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
                    const bool ng = (bc == BC_D) && (m & 1);           // Dirichlet: Y'_m = (-1)^m S_{N-1-m}
                    const double2 a = neg_if(v[q], ng), b = neg_if(v[q + E / 2], ng);
                    const double2 wm = ptw_rot<E>(w0, q, ptw, m);
                    v[q] = cmul(cconj(wm), make_double2(a.x + b.y, a.y - b.x));
                    if (m > 0) {                           // conj(w_{N-m}) = i w_m
                        smem[lay(N - m)] = cmul(make_double2(-wm.y, wm.x), make_double2(b.x + a.y, b.y - a.x));
                    } else {
                        const double2 h2 = dscale((bc == BC_N) ? 1.0 : sgn_of(H), yh);
                        constexpr double c4 = 0.70710678118654752440;          // conj(w_{N/2}) = c4 (1 + i)
                        smem[lay(H)] = make_double2(c4 * ((h2.x + h2.y) - (h2.y - h2.x)), c4 * ((h2.x + h2.y) + (h2.y - h2.x)));
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

    if constexpr (TSTORE) {
        // every exchange of the transform ended with a barrier: the tile buffer is free.  The un-permutation
        // is the permutation of the forward pass's loads: same positions.
#pragma unroll
        for (int q = 0; q < E; ++q) {
            const int i = t + q * P;
            const int pos = (bc == BC_P) ? i : ((bc == BC_N) ? ((i < H) ? i : H + (N - 1 - i)) : ((i < H) ? H + (H - 1 - i) : i - H));
            smem[pos * T + c] = (bc == BC_D) ? neg_if(v[q], i < H) : v[q];      // Dirichlet: x_{N-1-p} = -(-1)^p x'_p, p even for i < H
        }
        return;
    }
    if (!active) return;
#pragma unroll
    for (int q = 0; q < E; ++q) {
        const int i = t + q * P;
        if (bc == BC_P) {
            base[i * ld] = v[q];
        } else {
            const int p = (i < H) ? 2 * i : 2 * (N - 1 - i) + 1;
            if (bc == BC_N) base[p * ld] = v[q];
            else            base[(N - 1 - p) * ld] = neg_if(v[q], !(p & 1));      // x_{N-1-p} = -(-1)^p x'_p
        }
    }
}


template <int N>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
ypass_inv_kernel(double2 *w, int nxh, int bc, int complex_cols,
                 const double2 *__restrict__ tw, const double2 *__restrict__ ptw) {
    extern __shared__ double2 smem[];
    y_prefetch_ahead<N>(w, nxh, false);
    yinv_tile<N>(w, nxh, bc, complex_cols, tw, ptw, blockIdx.x, blockIdx.y, smem);
}

// slab decomposition: loads every row from the pencil block of the rank that owns it, stores the local z-slab w
template <int N>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
ypass_inv_slab_kernel(double2 *w, int nxh, int bc, int complex_cols,
                      const double2 *__restrict__ tw, const double2 *__restrict__ ptw, const __grid_constant__ YRows rows) {
    extern __shared__ double2 smem[];
    yinv_tile<N, true>(w, nxh, bc, complex_cols, tw, ptw, blockIdx.x, blockIdx.y, smem, &rows);
}

// Persistent staged kernels: CTA b transforms tiles b, b + gridDim.x, ... (tile = column tile bx of plane z, bx
// fastest: the resident CTAs work on neighbouring row segments of the same planes).  smem: the exchange scratch
// of the plain kernels, then the staging buffer.
template <int N, bool FWD_DIR>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YStaged<N>::PER_SM)
ypass_staged_kernel(double2 *w, int nxh, int nz, int bc, int complex_cols,
                    const double2 *__restrict__ tw, const double2 *__restrict__ ptw) {
    extern __shared__ double2 smem[];
    double2 *stage = smem + YCfg<N>::SMEM / sizeof(double2);
    constexpr int T = YCfg<N>::T;
    const int ntx = (nxh + T - 1) / T, total = ntx * nz;
    // forward: planes from the last to the first (the x pass before it left its last planes in L2)
    const auto plane_of = [&](int tile) { return FWD_DIR ? nz - 1 - tile / ntx : tile / ntx; };
    const auto issue = [&](int tile) {
        if (FWD_DIR) yfwd_stage_issue<N>(w, nxh, bc, tile % ntx, plane_of(tile), stage);
        else         yinv_stage_issue<N>(w, nxh, tile % ntx, plane_of(tile), stage);
    };
    int tile = blockIdx.x;
    if (tile < total) issue(tile);
    for (; tile < total; tile += gridDim.x) {
        cp_async_wait_all();
        __syncthreads();                           // the staged tile is complete; the previous tile is done with smem
        const int next = tile + (int)gridDim.x;
        const auto after_load = [&]() {
            __syncthreads();                       // every thread has read its part of the staging buffer
            if (next < total) issue(next);
        };
        if (FWD_DIR) yfwd_tile<N, false, false, 1>(w, nxh, bc, complex_cols, tw, ptw, tile % ntx, plane_of(tile), smem, nullptr, stage, after_load);
        else         yinv_tile<N, false, 1>(w, nxh, bc, complex_cols, tw, ptw, tile % ntx, plane_of(tile), smem, nullptr, stage, after_load);
    }
}


// ---- TMA-staged tiles (north_star item 3) -------------------------------------------------------------------
// Used where the row segments are narrow (N = 2048: T = 2, 32 bytes): a warp-wide 16-byte load then touches 16 lines,
// and the L1 tag stage -- one line per cycle -- costs more LSU cycles than all of the transform's shared-memory traffic
// (DESIGN.md section 6).  Here the copy engine fetches the tile instead: one thread issues N / 256 box copies
// (cp.async.bulk.tensor.3d, 256 rows x T*16 bytes each) into the CTA's tile buffer and everybody waits on the mbarrier;
// the threads then read their elements from shared memory (0.125 instead of 0.5 LSU cycles per element) and the SAME
// buffer becomes the exchange scratch -- no second buffer, the two resident CTAs per SM stay.  Stores are unchanged.
struct YTmaMaps {
    CUtensorMap all;      // every row of a plane: periodic forward pass, every inverse pass
    CUtensorMap even;     // rows 0, 2, 4, ...   (Neumann / Dirichlet forward pass)
    CUtensorMap odd;      // rows 1, 3, 5, ...
};
// rows per box: the tensor-map limit of 256, or 128 where 256 does not divide half the column (N = 1280)
__host__ __device__ constexpr int y_tma_box_rows(int n) { return (n / 2) % 256 == 0 ? 256 : 128; }

struct SyncHook {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};

template <int N>
__device__ __forceinline__ void y_tma_fetch(const YTmaMaps &maps, bool permuted, int bx, int z, double2 *tile, uint64_t *bar) {
    constexpr int T = YCfg<N>::T, Y_TMA_BOX_ROWS = y_tma_box_rows(N);
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_expect_tx(bar, (unsigned)(N * T * sizeof(double2)));
        if (!permuted) {
#pragma unroll
            for (int r = 0; r < N; r += Y_TMA_BOX_ROWS) tma_load_3d(tile + r * T, &maps.all, bx * T * 2, r, z, bar);
        } else {
#pragma unroll
            for (int r = 0; r < N / 2; r += Y_TMA_BOX_ROWS) {
                tma_load_3d(tile + r * T, &maps.even, bx * T * 2, r, z, bar);
                tma_load_3d(tile + (N / 2 + r) * T, &maps.odd, bx * T * 2, r, z, bar);
            }
        }
    }
    __syncthreads();                   // the barrier is initialised before anybody waits on it
    mbar_wait(bar, 0);
}

template <int N>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
ypass_fwd_tma_kernel(double2 *w, int nxh, int bc, int complex_cols, const double2 *__restrict__ tw,
                     const double2 *__restrict__ ptw, const __grid_constant__ YTmaMaps maps) {
    extern __shared__ __align__(128) double2 smem[];
    __shared__ __align__(8) uint64_t bar;
    const int z = gridDim.y - 1 - blockIdx.y;
    y_tma_fetch<N>(maps, bc != BC_P, blockIdx.x, z, smem, &bar);
    yfwd_tile<N, false, false, 2, SyncHook>(w, nxh, bc, complex_cols, tw, ptw, blockIdx.x, z, smem, nullptr, smem, SyncHook());
}

// the tile buffer -> global memory by the copy engine (rows as y_tma_fetch lays them out); the CTA leaves when the
// engine has read the buffer
template <int N>
__device__ __forceinline__ void y_tma_flush(const YTmaMaps &maps, bool permuted, int bx, int z, const double2 *tile) {
    constexpr int T = YCfg<N>::T, Y_TMA_BOX_ROWS = y_tma_box_rows(N);
    fence_proxy_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
        if (!permuted) {
#pragma unroll
            for (int r = 0; r < N; r += Y_TMA_BOX_ROWS) tma_store_3d(&maps.all, bx * T * 2, r, z, tile + r * T);
        } else {
#pragma unroll
            for (int r = 0; r < N / 2; r += Y_TMA_BOX_ROWS) {
                tma_store_3d(&maps.even, bx * T * 2, r, z, tile + r * T);
                tma_store_3d(&maps.odd, bx * T * 2, r, z, tile + (N / 2 + r) * T);
            }
        }
        tma_store_commit_and_wait_read();
    }
}

#ifndef PP_Y_TMA_STORE
#define PP_Y_TMA_STORE 0          // 1: the inverse pass's result leaves through the copy engine too.  Measured: no gain at
#endif                            // N = 2048 (3.94 against 3.91 TB/s), -7 % at 1024: the CTA then ends with a wait for the engine

template <int N>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
ypass_inv_tma_kernel(double2 *w, int nxh, int bc, int complex_cols, const double2 *__restrict__ tw,
                     const double2 *__restrict__ ptw, const __grid_constant__ YTmaMaps maps) {
    extern __shared__ __align__(128) double2 smem[];
    __shared__ __align__(8) uint64_t bar;
    y_tma_fetch<N>(maps, false, blockIdx.x, blockIdx.y, smem, &bar);
    yinv_tile<N, false, 1, SyncHook, PP_Y_TMA_STORE != 0>(w, nxh, bc, complex_cols, tw, ptw, blockIdx.x, blockIdx.y, smem, nullptr, smem, SyncHook());
    if (PP_Y_TMA_STORE) y_tma_flush<N>(maps, bc != BC_P, blockIdx.x, blockIdx.y, smem);
}

#ifndef PP_Y_TMA_MIN
#define PP_Y_TMA_MIN 1024         // y pass: TMA-staged tiles from this length on (measured: +1-7 % at 1024,
                                  // +7-13 % at 2048, -5 % at 512 where 128-byte row segments make the plain loads cheap)
#endif
template <int N>
struct YTma {
    static constexpr bool ON = (N >= PP_Y_TMA_MIN) && ((N / 2) % y_tma_box_rows(N) == 0);
};

}  // namespace pp
