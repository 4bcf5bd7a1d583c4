// x-pass kernels: the transform along the contiguous x axis, forward (first pass of the solve)
// and inverse (last pass), with the boundary-condition pre/post-processing fused in
// ("pre-processing / complex FFT / post-processing").
//
// Two real rows (2p, 2p+1 of the ny*nz rows) ride one complex FFT, z = a + i b; the Hermitian
// symmetry of a real signal's spectrum ("Enforce Hermitian symmetry") separates
// them afterwards:  A_m = (Z_m + conj Z_{N-m})/2,  B_m = (Z_m - conj Z_{N-m})/(2i).
//
//   periodic  (eq. 6)   packed half spectrum in N doubles per row:
//             [Re X_0, Re X_{N/2}, Re X_1, Im X_1, ..., Re X_{N/2-1}, Im X_{N/2-1}]
//   Neumann   (eq. 7, DCT-II)         Makhoul: v_i = z_{2i}, v_{N-1-i} = z_{2i+1},
//             Y_m = Re(w^m V_m), Y_{N-m} = -Im(w^m V_m), w = exp(-i pi/2N)
//   Dirichlet (eq. 9, DST-II)         the same around the wrapper [u5,-u4,u3,-u2,u1] on input and
//             output
// Inverse transforms (eq. 8 / eq. 10): V_m = conj(w)^m (Y_m - i Y_{N-m}),
// Y_N = 0, inverse FFT, un-permute.  All unnormalised; 1/(nx ny) is applied in the z solve.
#pragma once
#include "pp_fft.cuh"

namespace pp {

constexpr int BC_P = 0, BC_N = 1, BC_D = 2;

struct LayoutLin {
    __device__ __forceinline__ int operator()(int i) const { return pad8(i); }
};
// The partner exchange of the forward pass's post-processing (element m <-> N-m) goes through the same
// scratch UNPADDED: a quarter-warp then touches eight consecutive 16-byte slots in ascending or descending order --
// conflict-free either way -- where the padded layout puts the pad slot inside a descending run (two-way conflicts:
// ncu counted 3.5 M per x pass at 512 x 512 x 256, 12-14 % of its shared-memory wavefronts).  Measured: forward x pass
// +2 % at 512, +3-4 % at 1024 and 2048.
struct LayoutHand {
    __device__ __forceinline__ int operator()(int i) const { return i; }
};

// synchronise the P threads of one transform inside a CTA of T transforms
template <int P, int T>
struct GroupSync {
    int id;   // transform index within the CTA
    __device__ __forceinline__ void operator()() const {
        if constexpr (P >= 64 && T > 1 && T <= 15) {
            asm volatile("bar.sync %0, %1;" ::"r"(id + 1), "n"(P) : "memory");
        } else if constexpr (P <= 32 && (P * T) % 32 == 0) {
            __syncwarp();
        } else {
            __syncthreads();
        }
    }
};

__device__ __forceinline__ double sgn_of(int i) { return (i & 1) ? -1.0 : 1.0; }

#ifndef PP_X_MINB
#define PP_X_MINB 4
#endif

#ifndef PP_X_E16_MIN
#define PP_X_E16_MIN 4096     // x pass: 16 elements per thread from this length on (4096: never)
#endif

#ifndef PP_XI_E16_MIN
#define PP_XI_E16_MIN 1024    // inverse x pass: 16 elements per thread from this length on (one exchange fewer: measured
                              // +5 % at 1024 and 2048, where the forward pass loses with it)
#endif

template <int N, bool INVERSE = false>
struct XCfg {
    static constexpr int E = fft_E(N, INVERSE ? PP_XI_E16_MIN : PP_X_E16_MIN);
    using F = FftCfg<N, E>;
    static constexpr int P = F::P;
    static constexpr int T = (256 / P) > 0 ? (256 / P) : 1;   // transforms (row pairs) per CTA; <= 4 when P >= 64
    static constexpr int THREADS = T * P;
    // 8 elements per thread fit 64 registers (four CTAs per SM); 12 need about 80 (three CTAs: at 64 the 3 * 2^k
    // passes spilled up to 300 bytes per thread), 16 or 20 more than that
    static constexpr int MINB = (E <= 8) ? PP_X_MINB : ((E == 12) ? 3 : 2);
    static constexpr size_t SMEM = size_t(T) * F::SMEM_STRIDE * sizeof(double2);
};

// ------------------------------------------------------------------------------------------
// forward: real rows -> spectral rows
// ------------------------------------------------------------------------------------------
// One CTA-wide tile of the forward x pass: T row pairs starting at pair0, P threads each
// (blockDim.x == T * P).  `smem` holds T * FftCfg<N>::SMEM_ELEMS double2.
template <int N, int T>
__device__ __forceinline__ void xfwd_tile(const double *in, double *out, long long pair0, long long npairs, int bc,
                                          const double2 *__restrict__ tw, const double2 *__restrict__ ptw,
                                          double2 *smem) {
    using C = typename XCfg<N>::F;
    constexpr int E = C::E, P = C::P, H = N / 2;
    const int f = threadIdx.x / P, t = threadIdx.x % P;
    const long long pair = pair0 + f;
    const bool active = pair < npairs;
    const long long row = active ? pair * 2 : 0;
    const double *ra = in + row * N, *rb = ra + N;
    double *oa = out + row * N, *ob = oa + N;
    double2 *s = smem + f * C::SMEM_STRIDE;
    const LayoutLin lay;
    const LayoutHand hand;
    const GroupSync<P, T> sync{f};

    // ---- pre-processing fused into the load
    double2 v[E];
#pragma unroll
    for (int q = 0; q < E; ++q) {
        const int i = t + q * P;
        if (bc == BC_P) {
            v[q] = make_double2(ra[i], rb[i]);
        } else if (bc == BC_N) {
            const int p = (i < H) ? 2 * i : 2 * (N - 1 - i) + 1;
            v[q] = make_double2(ra[p], rb[p]);
        } else {
            // z'_m = (-1)^m z_{N-1-m}, then the Makhoul permutation
            if (i < H) { const int p = N - 1 - 2 * i; v[q] = make_double2(ra[p], rb[p]); }
            else       { const int p = 2 * i - N;     v[q] = make_double2(-ra[p], -rb[p]); }
        }
    }

    fft<N, FWD>(v, t, s, tw, lay, sync);

    // ---- post-processing: Hermitian separation of the two rows, twiddle, store.  The partner
    // Z_{N-m} of m in (0, N/2) lives in the upper half, so only that half goes through shared memory.
#pragma unroll
    for (int q = E / 2; q < E; ++q) s[hand(t + q * P)] = v[q];
    sync();
    if (active) {
        // the partners first, all in flight together, and one post-twiddle per thread (ptw_rot): loads issued
        // between the stores below queue behind them
        double2 zcs[E / 2];
        const double2 w0 = (bc != BC_P) ? __ldg(&ptw[t]) : make_double2(1.0, 0.0);
#pragma unroll
        for (int q = 0; q < E / 2; ++q) if (E >= PP_HOIST_ZC_MIN_E) zcs[q] = s[hand(neg_mod<N>(t + q * P))];
#pragma unroll
        for (int q = 0; q < E / 2; ++q) {
            const int m = t + q * P;                       // 0 <= m < N/2
            const double2 zm = v[q];
            const double2 zc = (E >= PP_HOIST_ZC_MIN_E) ? zcs[q] : s[hand(neg_mod<N>(m))];
            if (m == 0) {
                const double2 zh = v[E / 2];               // thread 0 also holds Z_{N/2}
                if (bc == BC_P) {
                    *reinterpret_cast<double2 *>(oa) = make_double2(zm.x, zh.x);
                    *reinterpret_cast<double2 *>(ob) = make_double2(zm.y, zh.y);
                } else {
                    constexpr double c4 = 0.70710678118654752440;   // cos(pi/4) = Re w_{N/2}
                    if (bc == BC_N) {
                        oa[0] = zm.x; ob[0] = zm.y;
                        oa[H] = c4 * zh.x; ob[H] = c4 * zh.y;
                    } else {                               // logical m -> N-1-m, sign -(-1)^m
                        oa[N - 1] = -zm.x; ob[N - 1] = -zm.y;
                        const double sg = -sgn_of(H);
                        oa[N - 1 - H] = sg * c4 * zh.x; ob[N - 1 - H] = sg * c4 * zh.y;
                    }
                }
            } else {
                const double2 A = make_double2(0.5 * (zm.x + zc.x), 0.5 * (zm.y - zc.y));
                const double2 B = make_double2(0.5 * (zm.y + zc.y), -0.5 * (zm.x - zc.x));
                if (bc == BC_P) {
                    *reinterpret_cast<double2 *>(oa + 2 * m) = A;
                    *reinterpret_cast<double2 *>(ob + 2 * m) = B;
                } else {
                    const double2 w = ptw_rot<E>(w0, q, ptw, m);
                    const double2 ca = cmul(w, A), cb = cmul(w, B);
                    if (bc == BC_N) {
                        oa[m] = ca.x;      ob[m] = cb.x;
                        oa[N - m] = -ca.y; ob[N - m] = -cb.y;
                    } else {
                        const bool odd = m & 1;                        // logical m: sign -(-1)^m
                        oa[N - 1 - m] = neg_if(ca.x, !odd); ob[N - 1 - m] = neg_if(cb.x, !odd);
                        // logical N-m -> position m-1: -Im with sign -(-1)^(N-m) = -(-1)^m, i.e. (-1)^m Im
                        oa[m - 1] = neg_if(ca.y, odd);      ob[m - 1] = neg_if(cb.y, odd);
                    }
                }
            }
        }
    }
}


template <int N>
__global__ void __launch_bounds__(XCfg<N>::THREADS, XCfg<N>::MINB)
xpass_fwd_kernel(const double *in, double *out, long long npairs, int bc,
                 const double2 *__restrict__ tw, const double2 *__restrict__ ptw) {
    extern __shared__ double2 smem[];
    xfwd_tile<N, XCfg<N>::T>(in, out, (long long)blockIdx.x * XCfg<N>::T, npairs, bc, tw, ptw, smem);
}

// ------------------------------------------------------------------------------------------
// inverse: spectral rows -> real rows
// ------------------------------------------------------------------------------------------
// One CTA-wide tile of the inverse x pass (see xfwd_tile).  LDCG: read the input with ld.global.cg
// (L2 only) -- for the fused y+x kernel, whose input rows were just written by other SMs.
template <bool LDCG>
__device__ __forceinline__ double xld(const double *p) { return LDCG ? __ldcg(p) : *p; }
template <bool LDCG>
__device__ __forceinline__ double2 xld2(const double *p) {
    return LDCG ? __ldcg(reinterpret_cast<const double2 *>(p)) : *reinterpret_cast<const double2 *>(p);
}

template <int N, int T, bool LDCG>
__device__ __forceinline__ void xinv_tile(const double *in, double *out, long long pair0, long long npairs, int bc,
                                          const double2 *__restrict__ tw, const double2 *__restrict__ ptw,
                                          double2 *smem) {
    using C = typename XCfg<N, true>::F;
    constexpr int E = C::E, P = C::P, H = N / 2;
    const int f = threadIdx.x / P, t = threadIdx.x % P;
    const long long pair = pair0 + f;
    const bool active = pair < npairs;
    const long long row = active ? pair * 2 : 0;
    const double *ra = in + row * N, *rb = ra + N;
    double *oa = out + row * N, *ob = oa + N;
    double2 *s = smem + f * C::SMEM_STRIDE;
    const LayoutLin lay;
    const LayoutLin hand;      // the inverse pass keeps the padded layout for its hand-offs (unpadded measured 3 % slower at 16 elements per thread)
    const GroupSync<P, T> sync{f};

    double2 v[E];
    if (bc == BC_P) {
        // Every packed element (A_m, B_m), m in [0, N/2), is loaded once by the thread that owns Z_m;
        // the mirrored Z_{N-m} = conj(A_m) + i conj(B_m) is handed to its owner through shared memory.
#pragma unroll
        for (int q = 0; q < E / 2; ++q) {
            const int m = t + q * P;
            const double2 A = xld2<LDCG>(ra + 2 * m);
            const double2 B = xld2<LDCG>(rb + 2 * m);
            if (m == 0) {                                              // (X_0, X_{N/2}) of both rows, all real
                v[q] = make_double2(A.x, B.x);
                s[hand(H)] = make_double2(A.y, B.y);
            } else {
                v[q] = make_double2(A.x - B.y, A.y + B.x);             // Z_m = A + i B
                s[hand(N - m)] = make_double2(A.x + B.y, B.x - A.y);    // Z_{N-m}
            }
        }
    } else {
        // Neumann / Dirichlet: V_m = conj(w_m) (Y_m - i Y_{N-m}) and V_{N-m} = conj(w_{N-m}) (Y_{N-m} - i Y_m)
        // need the same two coefficients, and conj(w_{N-m}) = i w_m.  The owner of m in [0, N/2) loads the
        // pair once, keeps V_m and hands V_{N-m} to its owner through shared memory, exactly as above.
        // Packed rows: Y = Ya + i Yb, so Y_m - i Y_{N-m} = (ya + ybp) + i (yb - yap).
        // (all loads first, so that they are in flight together; then the arithmetic)
        double la[E / 2], lb[E / 2], lap[E / 2], lbp[E / 2], ha = 0.0, hb = 0.0;
        const double2 w0 = __ldg(&ptw[t]);                 // the other pre-twiddles by rotation (ptw_rot)
#pragma unroll
        for (int q = 0; q < E / 2; ++q) {
            const int m = t + q * P;
            const int at = (bc == BC_N) ? m : N - 1 - m, atp = (bc == BC_N) ? N - m : m - 1;
            la[q] = xld<LDCG>(ra + at); lb[q] = xld<LDCG>(rb + at);
            lap[q] = (m > 0) ? xld<LDCG>(ra + atp) : 0.0;
            lbp[q] = (m > 0) ? xld<LDCG>(rb + atp) : 0.0;
            if (m == 0) {                                              // thread 0 also makes V_{N/2} (its own partner)
                const int ah = (bc == BC_N) ? H : N - 1 - H;
                ha = xld<LDCG>(ra + ah); hb = xld<LDCG>(rb + ah);
            }
        }
#pragma unroll
        for (int q = 0; q < E / 2; ++q) {
            const int m = t + q * P;
            const bool ng = (bc == BC_D) && (m & 1);                   // Dirichlet: Y'_m = (-1)^m S_{N-1-m}
            const double ya = neg_if(la[q], ng), yb = neg_if(lb[q], ng), yap = neg_if(lap[q], ng), ybp = neg_if(lbp[q], ng);
            const double2 w = ptw_rot<E>(w0, q, ptw, m);
            v[q] = cmul(cconj(w), make_double2(ya + ybp, yb - yap));
            if (m > 0) {
                s[hand(N - m)] = cmul(make_double2(-w.y, w.x), make_double2(yap + yb, ybp - ya));   // i w_m (...)
            } else {
                const double sh = (bc == BC_N) ? 1.0 : sgn_of(H);
                constexpr double c4 = 0.70710678118654752440;              // conj(w_{N/2}) = c4 (1 + i)
                const double hr = sh * (ha + hb), hi = sh * (hb - ha);
                s[hand(H)] = make_double2(c4 * (hr - hi), c4 * (hr + hi));
            }
        }
    }
    // every load of this row pair precedes the barrier, every store follows it: in-place safe
    sync();
#pragma unroll
    for (int q = E / 2; q < E; ++q) v[q] = s[hand(t + q * P)];
    sync();

    fft<N, INV>(v, t, s, tw, lay, sync);

    if (bc == BC_P) {
        if (active) {
#pragma unroll
            for (int q = 0; q < E; ++q) { oa[t + q * P] = v[q].x; ob[t + q * P] = v[q].y; }
        }
        return;
    }
    // Neumann / Dirichlet: the un-permutation sends v_i to position 2i and v_{N-1-i} to
    // 2i+1 (i < N/2) -- neighbours.  The upper half goes through shared memory to the owner of i, which
    // stores both as one 16-byte element instead of two 8-byte ones at stride 2.
#pragma unroll
    for (int q = E / 2; q < E; ++q) s[hand(t + q * P)] = v[q];
    sync();
    if (active) {
#pragma unroll
        for (int q = 0; q < E / 2; ++q) {
            const int i = t + q * P;                                   // 0 <= i < N/2
            const double2 lo = v[q], hi = s[hand(N - 1 - i)];
            if (bc == BC_N) {
                *reinterpret_cast<double2 *>(oa + 2 * i) = make_double2(lo.x, hi.x);
                *reinterpret_cast<double2 *>(ob + 2 * i) = make_double2(lo.y, hi.y);
            } else {                                                   // x_{N-1-p} = -(-1)^p x'_p: (x_{N-2-2i}, x_{N-1-2i})
                *reinterpret_cast<double2 *>(oa + N - 2 - 2 * i) = make_double2(hi.x, -lo.x);
                *reinterpret_cast<double2 *>(ob + N - 2 - 2 * i) = make_double2(hi.y, -lo.y);
            }
        }
    }
}

template <int N>
__global__ void __launch_bounds__(XCfg<N, true>::THREADS, XCfg<N, true>::MINB)
xpass_inv_kernel(const double *in, double *out, long long npairs, int bc,
                 const double2 *__restrict__ tw, const double2 *__restrict__ ptw) {
    extern __shared__ double2 smem[];
    // rows from the last to the first: the y pass before this one went plane 0 to plane nz-1, so its
    // last planes are still in L2
    xinv_tile<N, XCfg<N, true>::T, false>(in, out, (long long)(gridDim.x - 1 - blockIdx.x) * XCfg<N, true>::T, npairs, bc, tw, ptw, smem);
}

}  // namespace pp
