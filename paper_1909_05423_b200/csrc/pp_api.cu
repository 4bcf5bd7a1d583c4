// C ABI of pittpack_b200 (include/pittpack_b200.h): plan construction, table generation and the
// five-kernel solve.  No cuFFT / cuSPARSE, no CPU fallback.
#include "../../include/pittpack_b200.h"

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "pp_fft.cuh"
#include "pp_xpass.cuh"
#include "pp_ypass.cuh"
#include "pp_zsolve.cuh"
#include "pp_zpart.cuh"
#include "pp_fused.cuh"

using namespace pp;

struct pp_plan {
    int nx, ny, nz;
    double dx, dy, dz;
    int bcx, bcy, bcz;
    int device;
    int num_sms;
    int singular;
    double scale;
    double2 *tw_x, *tw_y;      // per-stage FFT twiddle tables (pp_fft.cuh, tw_stage_offset)
    double2 *ptw_x, *ptw_y;    // exp(-i pi m / (2n)), m in [0, n]
    double *sx, *sy;           // dz^2 lam / h^2 per packed position
    double *zero_scratch;      // [nz]
    double *host_stage;        // N doubles, created by the first pp_solve_host
    // pp_solve_host_batch: a ring of staging buffers, a copy-in and a copy-out stream, events per buffer
    static constexpr int NSTAGE = 3;
    double *batch_stage[NSTAGE];
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_in[NSTAGE], ev_done[NSTAGE], ev_out[NSTAGE];
    size_t bytes;
    int profiling;
    int have_times;
    int z_algorithm;           // PP_Z_AUTO / PP_Z_SWEEP / PP_Z_PARTITION
    double bmax;               // largest |diagonal| of any z system, 3 + max |s| (range check of the partitioned kernels)
    int null_space;            // PP_NULL_ZERO_MEAN / PP_NULL_PIN_PLANE0 (singular problems only)
    int xy_fusion;             // 1: x and y passes of a plane run as tasks of one kernel (pp_fused.cuh)
    int *fuse_sync;            // [1 + nz] ticket + per-plane completion counters
    double *hier_scratch;      // [4][nz / 256][nx ny]: interface values of the two-level z solve (long lines only)
    cudaStream_t side;         // long singular lines only: the zero-mode line is solved beside the two-level passes
    cudaEvent_t ev_fork, ev_join;
    cudaEvent_t ev[PP_NUM_KERNELS + 1];
};

// ------------------------------------------------------------------------------------------
// host-side tables, evaluated in long double and rounded once
// ------------------------------------------------------------------------------------------
namespace {

const long double PI_L = 3.14159265358979323846264338327950288L;

// powers of two in [4, 2048], 3 * 2^k in [48, 1536], 5 * 2^k in [80, 1280]
bool length_supported(int n) { return n >= 4 && n <= 2048 && fft_length_ok(n); }

void make_twiddles(int n, std::vector<double2> &tw, std::vector<double2> &ptw) {
    tw.assign(tw_table_elems(n), make_double2(1.0, 0.0));
    ptw.resize(n + 1);
    // stage with NS: row r = 1 (radix 8) or rows r = 1, 2 (radix 4) of W_n^(k r stride), stride = n / (RS NS), k in [0, NS)
    const int rs = stage_radix(n), rows = tw_rows(n);
    for (int ns = first_radix(n); ns < n; ns *= rs) {
        const int off = tw_stage_offset(n, ns), stride = n / (rs * ns);
        for (int ri = 0; ri < rows; ++ri)
            for (int k = 0; k < ns; ++k) {
                const long long e = ((long long)k * (1 << ri) * stride) % n;
                const long double a = 2.0L * PI_L * (long double)e / (long double)n;
                tw[off + ri * ns + k] = make_double2((double)cosl(a), (double)(-sinl(a)));
            }
    }
    for (int m = 0; m <= n; ++m) {
        const long double a = PI_L * (long double)m / (2.0L * (long double)n);
        ptw[m] = make_double2((double)cosl(a), (double)(-sinl(a)));
    }
}

// Table 2: modified wavenumber of wavenumber index k on an axis of length n.
long double table2(int bc, int k, int n) {
    long double arg;
    if (bc == PP_BC_PERIODIC) arg = 2.0L * PI_L * (long double)k / (long double)n;
    else if (bc == PP_BC_NEUMANN) arg = PI_L * (long double)k / (long double)n;
    else arg = PI_L * (long double)(k + 1) / (long double)n;
    const long double sh = sinl(0.5L * arg);
    return -4.0L * sh * sh;                      // = -2 + 2 cos(arg), without the cancellation
}

// shift table per stored position: `packed_x` = the x-pass layout (periodic: [X_0, X_n/2, Re X_1, Im X_1, ..]),
// otherwise position == wavenumber index (also for half-complex periodic rows: lam is even in k).
void make_shift(int bc, int n, bool packed_x, long double factor, std::vector<double> &s) {
    s.resize(n);
    for (int p = 0; p < n; ++p) {
        int k = p;
        if (bc == PP_BC_PERIODIC && packed_x) k = (p == 0) ? 0 : ((p == 1) ? n / 2 : p / 2);
        s[p] = (double)(factor * table2(bc, k, n));
    }
}

template <class T>
int upload(T **dst, const std::vector<T> &src, size_t &bytes) {
    const size_t nb = src.size() * sizeof(T);
    if (cudaMalloc((void **)dst, nb) != cudaSuccess) { *dst = nullptr; cudaGetLastError(); return PP_ERR_ALLOC; }
    bytes += nb;
    if (cudaMemcpy(*dst, src.data(), nb, cudaMemcpyHostToDevice) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    return PP_SUCCESS;
}

// ------------------------------------------------------------------------------------------
// launch helpers
// ------------------------------------------------------------------------------------------
template <class K>
int set_smem(K kernel, size_t smem) {
    if (smem > 48 * 1024) {
        if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
            cudaGetLastError();
            return PP_ERR_CUDA;
        }
    }
    return PP_SUCCESS;
}

template <int N>
int launch_x(bool fwd, const double *in, double *out, long long npairs, int bc, const double2 *tw,
             const double2 *ptw, cudaStream_t st) {
    using X = XCfg<N>;
    const unsigned grid = (unsigned)((npairs + X::T - 1) / X::T);
    auto kf = xpass_fwd_kernel<N>;
    auto ki = xpass_inv_kernel<N>;
    if (int rc = set_smem(fwd ? kf : ki, X::SMEM)) return rc;
    if (fwd) kf<<<grid, X::THREADS, X::SMEM, st>>>(in, out, npairs, bc, tw, ptw);
    else     ki<<<grid, X::THREADS, X::SMEM, st>>>(in, out, npairs, bc, tw, ptw);
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}

template <int N>
int launch_y(bool fwd, double *w, int nxh, int nz, int bc, int complex_cols, const double2 *tw,
             const double2 *ptw, cudaStream_t st) {
    using Y = YCfg<N>;
    const dim3 grid((unsigned)((nxh + Y::T - 1) / Y::T), (unsigned)nz);
    auto kf = ypass_fwd_kernel<N>;
    auto ki = ypass_inv_kernel<N>;
    if (int rc = set_smem(fwd ? kf : ki, Y::SMEM)) return rc;
    if (fwd) kf<<<grid, Y::THREADS, Y::SMEM, st>>>((double2 *)w, nxh, bc, complex_cols, tw, ptw);
    else     ki<<<grid, Y::THREADS, Y::SMEM, st>>>((double2 *)w, nxh, bc, complex_cols, tw, ptw);
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}

#define PP_DISPATCH_N(n, CALL)                       \
    switch (n) {                                     \
        case 4:    return CALL(4);                   \
        case 8:    return CALL(8);                   \
        case 16:   return CALL(16);                  \
        case 32:   return CALL(32);                  \
        case 64:   return CALL(64);                  \
        case 128:  return CALL(128);                 \
        case 256:  return CALL(256);                 \
        case 512:  return CALL(512);                 \
        case 1024: return CALL(1024);                \
        case 2048: return CALL(2048);                \
        case 48:   return CALL(48);                  \
        case 96:   return CALL(96);                  \
        case 192:  return CALL(192);                 \
        case 384:  return CALL(384);                 \
        case 768:  return CALL(768);                 \
        case 1536: return CALL(1536);                \
        case 80:   return CALL(80);                  \
        case 160:  return CALL(160);                 \
        case 320:  return CALL(320);                 \
        case 640:  return CALL(640);                 \
        case 1280: return CALL(1280);                \
        default:   return PP_ERR_UNSUPPORTED_SIZE;   \
    }

int run_x(const pp_plan *p, bool fwd, const double *in, double *out, cudaStream_t st) {
    const long long npairs = (long long)p->ny * p->nz / 2;
#define CALL_X(NN) launch_x<NN>(fwd, in, out, npairs, p->bcx, p->tw_x, p->ptw_x, st)
    PP_DISPATCH_N(p->nx, CALL_X)
#undef CALL_X
}

int run_y(const pp_plan *p, bool fwd, double *w, cudaStream_t st) {
    const int complex_cols = (p->bcx == PP_BC_PERIODIC && p->bcy == PP_BC_PERIODIC) ? 1 : 0;
#define CALL_Y(NN) launch_y<NN>(fwd, w, p->nx / 2, p->nz, p->bcy, complex_cols, p->tw_y, p->ptw_y, st)
    PP_DISPATCH_N(p->ny, CALL_Y)
#undef CALL_Y
}

// The partitioned z kernels tabulate the leading minors q_0 .. q_R of a segment block, |q_R| <= bmax^R:
// for grids so anisotropic (dz >> dx) that this could leave the fp64 range they are not used.
bool zpart_range_ok(const pp_plan *p, int R) { return (double)R * std::log2(p->bmax) < 1000.0; }
ZPartShape plan_zpart_shape(const pp_plan *p) {
    const ZPartShape z = zpart_shape(p->nz);
    return (z.R && zpart_range_ok(p, z.R)) ? z : ZPartShape{0, 0, 0};
}

// Non-homogeneous Dirichlet face values moved to the right-hand side:
//   f[offset + i sf + j ss] -= coef g[j nf + i],   coef = 2 / h^2,  (i, j) over one face of nf x ns cells
__global__ void fold_face_kernel(double *f, const double *__restrict__ g, int nf, int ns, long long sf, long long ss,
                                 long long offset, double coef) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i < nf && j < ns) {
        double *cell = f + offset + i * sf + j * ss;
        *cell = *cell - __dmul_rn(coef, g[(long long)j * nf + i]);      // two roundings, like the oracle (no FMA)
    }
}

// nx == ny in {128, 256, 512, 1024}: the sizes the fused x+y kernel is instantiated for
bool fusion_supported(int nx, int ny) { return nx == ny && nx >= 128 && nx <= 1024 && (nx & (nx - 1)) == 0; }

#ifndef PP_FUSE_LAG
#define PP_FUSE_LAG 0          // 0: derived from the number of resident CTAs
#endif

template <int N, bool FWD_DIR>
int launch_fused(const pp_plan *p, const double *in, double *u, cudaStream_t st) {
    using Y = YCfg<N>;
    constexpr int TX = Y::THREADS / FftCfg<N>::P;
    auto kernel = xy_fused_kernel<N, FWD_DIR>;
    if (int rc = set_smem(kernel, Y::SMEM)) return rc;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, Y::THREADS, Y::SMEM) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        return PP_ERR_CUDA;
    }
    FusedParams fp;
    fp.nz = p->nz; fp.nxh = p->nx / 2;
    fp.pairs_per_plane = p->ny / 2;
    const int xt = (int)((fp.pairs_per_plane + TX - 1) / TX), yt = (fp.nxh + Y::T - 1) / Y::T;
    fp.na = FWD_DIR ? xt : yt;
    fp.nb = FWD_DIR ? yt : xt;
    const long long resident = (long long)p->num_sms * per_sm;
    long long lag = PP_FUSE_LAG ? PP_FUSE_LAG : (5 * resident / (4 * (fp.na + fp.nb)) + 2);
    fp.lag = (int)(lag < 1 ? 1 : (lag > p->nz ? p->nz : lag));
    fp.bcx = p->bcx; fp.bcy = p->bcy;
    fp.complex_cols = (p->bcx == PP_BC_PERIODIC && p->bcy == PP_BC_PERIODIC) ? 1 : 0;
    fp.sync = p->fuse_sync;
    if (cudaMemsetAsync(p->fuse_sync, 0, sizeof(int) * (size_t)(p->nz + 1), st) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    const long long total = (long long)p->nz * (fp.na + fp.nb);
    const unsigned grid = (unsigned)(total < resident ? total : resident);
    kernel<<<grid, Y::THREADS, Y::SMEM, st>>>(in, u, fp, p->tw_x, p->ptw_x, p->tw_y, p->ptw_y);
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}

int run_fused(const pp_plan *p, bool fwd, const double *in, double *u, cudaStream_t st) {
    switch (p->nx) {
        case 128:  return fwd ? launch_fused<128, true>(p, in, u, st) : launch_fused<128, false>(p, in, u, st);
        case 256:  return fwd ? launch_fused<256, true>(p, in, u, st) : launch_fused<256, false>(p, in, u, st);
        case 512:  return fwd ? launch_fused<512, true>(p, in, u, st) : launch_fused<512, false>(p, in, u, st);
        case 1024: return fwd ? launch_fused<1024, true>(p, in, u, st) : launch_fused<1024, false>(p, in, u, st);
        default:   return PP_ERR_UNSUPPORTED_SIZE;
    }
}

int run_z(const pp_plan *p, double *w, cudaStream_t st) {
    ZParams zp;
    zp.nx = p->nx; zp.ny = p->ny; zp.nz = p->nz;
    zp.bcz = p->bcz;
    zp.singular = p->singular ? (p->null_space == PP_NULL_PIN_PLANE0 ? 2 : 1) : 0;
    zp.scale = p->scale;
    zp.sx = p->sx; zp.sy = p->sy;
    zp.zero_scratch = p->zero_scratch;
    const size_t plane = (size_t)p->nx * p->ny;
#ifndef PP_Z_DSMEM
#define PP_Z_DSMEM 0
#endif
#ifndef PP_Z_CB
#define PP_Z_CB 16
#endif
    const bool want_part = p->z_algorithm != PP_Z_SWEEP;
    const ZPartShape zs = want_part ? plan_zpart_shape(p) : ZPartShape{0, 0, 0};
    if (zs.R) {
        // partitioned, register-resident solve: one HBM read + one write per unknown (pp_zpart.cuh)
        const bool cyc = p->bcz == PP_BC_PERIODIC;
        const size_t ds = zpart_smem_bytes(zs, cyc);
        const unsigned grid = (unsigned)((plane + zs.L - 1) / zs.L);
        const ZHier none = {1, nullptr, nullptr};
        auto launch = [&](auto kernel) -> int {
            if (int rc = set_smem(kernel, ds)) return rc;
            kernel<<<grid, zs.L * zs.S, ds, st>>>(w, zp, zs.S, zs.L, none);
            return PP_SUCCESS;
        };
        int rc;
        if (zs.R == 32) rc = cyc ? launch(zsolve_part_kernel<32, 0, true>) : launch(zsolve_part_kernel<32, 0, false>);
        else            rc = cyc ? launch(zsolve_part_kernel<64, 0, true>) : launch(zsolve_part_kernel<64, 0, false>);
        if (rc) return rc;
    } else if (want_part && p->hier_scratch) {
        // long lines: two-level partition, 8 + 16 bytes per unknown (pp_zpart.cuh, ZHier)
        const ZPartShape hs = {32, ZP_HIER_ROWS / 32, 32};
        const size_t ds = zpart_smem_bytes(hs);
        const int nK = p->nz / ZP_HIER_ROWS;
        const size_t slab = (size_t)nK * plane;
        const ZHier h = {nK, p->hier_scratch, p->hier_scratch + slab};
        const dim3 grid((unsigned)((plane + hs.L - 1) / hs.L), (unsigned)nK);
        if (int rc = set_smem(zsolve_part_kernel<32, 1>, ds)) return rc;
        if (int rc = set_smem(zsolve_part_kernel<32, 2>, ds)) return rc;
        if (p->singular) {
            // the singular (0,0) line touches column 0 only, which the passes below never store and whose
            // values they discard: it runs beside them on the plan's side stream (fork / join by events)
            if (cudaEventRecord(p->ev_fork, st) != cudaSuccess || cudaStreamWaitEvent(p->side, p->ev_fork, 0) != cudaSuccess) {
                cudaGetLastError();
                return PP_ERR_CUDA;
            }
            zero_mode_long_kernel<<<1, 1024, 0, p->side>>>(w, plane, p->nz, p->scale, p->null_space == PP_NULL_PIN_PLANE0);
            if (cudaEventRecord(p->ev_join, p->side) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
        }
        zsolve_part_kernel<32, 1><<<grid, hs.L * hs.S, ds, st>>>(w, zp, hs.S, hs.L, h);
        zsolve_hier_interface_kernel<<<(unsigned)((plane + 63) / 64), 64, 0, st>>>(zp, h, ZP_HIER_ROWS, p->hier_scratch + 2 * slab,
                                                                             p->hier_scratch + 3 * slab);
        zsolve_part_kernel<32, 2><<<grid, hs.L * hs.S, ds, st>>>(w, zp, hs.S, hs.L, h);
        if (p->singular && cudaStreamWaitEvent(st, p->ev_join, 0) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    } else if (p->bcz != PP_BC_PERIODIC) {
        // checkpoint table in shared memory: ceil(nz / CB) x TH doubles per CTA
#define PP_ZT_LAUNCH(C, T)                                                                           \
        do {                                                                                         \
            const size_t ds = (size_t)(((p->nz + 1) / 2 + C - 1) / C) * T * sizeof(double) + PP_Z_DSMEM; \
            if (int rc = set_smem(zsolve_thomas_kernel<C, T>, ds)) return rc;                        \
            zsolve_thomas_kernel<C, T><<<(unsigned)((plane + T - 1) / T), T, ds, st>>>(w, zp);       \
        } while (0)
#ifdef PP_Z_TH
        PP_ZT_LAUNCH(PP_Z_CB, PP_Z_TH);
#else
        PP_ZT_LAUNCH(PP_Z_CB, 128);
#endif
#undef PP_ZT_LAUNCH
    } else {
        constexpr int TH = PP_Z_THREADS;
        const unsigned grid = (unsigned)((plane + TH - 1) / TH);
        const int cb = (p->nz <= 16 * Z_MAX_CK) ? 16 : ((p->nz <= 32 * Z_MAX_CK) ? 32 : 64);
        const size_t ds = PP_Z_DSMEM;      // dummy dynamic shared memory: caps resident CTAs per SM
#define PP_Z_LAUNCH(K, C)                                                                        \
        do {                                                                                     \
            if (int rc = set_smem(K<C>, ds)) return rc;                                          \
            K<C><<<grid, TH, ds, st>>>(w, zp);                                                   \
        } while (0)
        if (cb == 16)      PP_Z_LAUNCH(zsolve_cyclic_kernel, 16);
        else if (cb == 32) PP_Z_LAUNCH(zsolve_cyclic_kernel, 32);
        else               PP_Z_LAUNCH(zsolve_cyclic_kernel, 64);
#undef PP_Z_LAUNCH
    }
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}

void free_plan(pp_plan *p) {
    if (!p) return;
    cudaFree(p->tw_x); cudaFree(p->tw_y); cudaFree(p->ptw_x); cudaFree(p->ptw_y);
    cudaFree(p->sx); cudaFree(p->sy); cudaFree(p->zero_scratch); cudaFree(p->host_stage); cudaFree(p->fuse_sync); cudaFree(p->hier_scratch);
    for (auto &e : p->ev) if (e) cudaEventDestroy(e);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->side) cudaStreamDestroy(p->side);
    for (int b = 0; b < pp_plan::NSTAGE; ++b) {
        cudaFree(p->batch_stage[b]);
        if (p->ev_in[b]) cudaEventDestroy(p->ev_in[b]);
        if (p->ev_done[b]) cudaEventDestroy(p->ev_done[b]);
        if (p->ev_out[b]) cudaEventDestroy(p->ev_out[b]);
    }
    if (p->s_in) cudaStreamDestroy(p->s_in);
    if (p->s_out) cudaStreamDestroy(p->s_out);
    cudaGetLastError();
    delete p;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------
extern "C" {

const char *pp_version(void) { return "pittpack_b200 0.1 (sm_100a)"; }

const char *pp_strerror(int status) {
    switch (status) {
        case PP_SUCCESS: return "success";
        case PP_ERR_INVALID_ARG: return "invalid argument";
        case PP_ERR_UNSUPPORTED_SIZE: return "unsupported grid size (nx, ny: 2^k in [4, 2048], 3*2^k in [48, 1536] or 5*2^k in [80, 1280]; nz in [2, 4096], or 256 m <= 16384 with non-periodic z)";
        case PP_ERR_ALLOC: return "allocation failed";
        case PP_ERR_CUDA: return "CUDA runtime or launch error (is a CUDA device present?)";
        case PP_ERR_NULL: return "null pointer argument";
        default: return "unknown status";
    }
}

int pp_plan_create(pp_plan **out, int nx, int ny, int nz, double dx, double dy, double dz,
                   int bc_x, int bc_y, int bc_z) {
    if (!out) return PP_ERR_NULL;
    *out = nullptr;
    if (nx <= 0 || ny <= 0 || nz <= 0) return PP_ERR_INVALID_ARG;
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz))
        return PP_ERR_INVALID_ARG;
    for (int bc : {bc_x, bc_y, bc_z})
        if (bc != PP_BC_PERIODIC && bc != PP_BC_NEUMANN && bc != PP_BC_DIRICHLET) return PP_ERR_INVALID_ARG;
    // nz: the two-sweep kernels take any nz up to 4096; longer lines need the two-level partition
    // (Neumann / Dirichlet z, nz a multiple of 256 up to 16384)
    const bool long_ok = bc_z != PP_BC_PERIODIC && zpart_hier_ok(nz);
    if (!length_supported(nx) || !length_supported(ny) || nz < 2 || (nz > 64 * Z_MAX_CK && !long_ok)) return PP_ERR_UNSUPPORTED_SIZE;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }

    pp_plan *p = new (std::nothrow) pp_plan();
    if (!p) return PP_ERR_ALLOC;
    std::memset(p, 0, sizeof(*p));
    p->nx = nx; p->ny = ny; p->nz = nz;
    p->dx = dx; p->dy = dy; p->dz = dz;
    p->bcx = bc_x; p->bcy = bc_y; p->bcz = bc_z;
    p->device = dev;
    if (cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || p->num_sms <= 0) {
        cudaGetLastError();
        delete p;
        return PP_ERR_CUDA;
    }
    p->singular = (bc_x != PP_BC_DIRICHLET && bc_y != PP_BC_DIRICHLET && bc_z != PP_BC_DIRICHLET) ? 1 : 0;
    p->scale = (double)((long double)dz * (long double)dz / ((long double)nx * (long double)ny));

    std::vector<double2> tw, ptw;
    std::vector<double> s;
    int rc = PP_SUCCESS;
    make_twiddles(nx, tw, ptw);
    if (!rc) rc = upload(&p->tw_x, tw, p->bytes);
    if (!rc) rc = upload(&p->ptw_x, ptw, p->bytes);
    make_twiddles(ny, tw, ptw);
    if (!rc) rc = upload(&p->tw_y, tw, p->bytes);
    if (!rc) rc = upload(&p->ptw_y, ptw, p->bytes);
    const long double dz2 = (long double)dz * (long double)dz;
    double smin = 0.0;
    make_shift(bc_x, nx, true, dz2 / ((long double)dx * (long double)dx), s);
    { double m = 0.0; for (double v : s) m = v < m ? v : m; smin += m; }
    if (!rc) rc = upload(&p->sx, s, p->bytes);
    make_shift(bc_y, ny, false, dz2 / ((long double)dy * (long double)dy), s);
    { double m = 0.0; for (double v : s) m = v < m ? v : m; smin += m; }
    if (!rc) rc = upload(&p->sy, s, p->bytes);
    p->bmax = 3.0 - smin;
    // lines beyond the two-sweep kernel's range need the two-level partition (segments of 32 rows)
    if (!rc && nz > 64 * Z_MAX_CK && !zpart_range_ok(p, 32)) rc = PP_ERR_UNSUPPORTED_SIZE;
    if (!rc) {
        std::vector<double> z((size_t)nz, 0.0);
        rc = upload(&p->zero_scratch, z, p->bytes);
    }
    if (!rc && long_ok && zpart_shape(nz).R == 0 && zpart_range_ok(p, 32)) {
        const size_t nb = sizeof(double) * 4 * (size_t)(nz / ZP_HIER_ROWS) * (size_t)nx * (size_t)ny;
        if (cudaMalloc((void **)&p->hier_scratch, nb) != cudaSuccess) { p->hier_scratch = nullptr; cudaGetLastError(); rc = PP_ERR_ALLOC; }
        else p->bytes += nb;
    }
    if (!rc && p->hier_scratch && p->singular) {
        if (cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            rc = PP_ERR_CUDA;
        }
    }
    if (!rc) {
        const size_t nb = sizeof(int) * (size_t)(nz + 1);
        if (cudaMalloc((void **)&p->fuse_sync, nb) != cudaSuccess) { p->fuse_sync = nullptr; cudaGetLastError(); rc = PP_ERR_ALLOC; }
        else p->bytes += nb;
    }
    if (!rc) {
        for (auto &e : p->ev)
            if (cudaEventCreate(&e) != cudaSuccess) { e = nullptr; cudaGetLastError(); rc = PP_ERR_CUDA; break; }
    }
    if (rc) { free_plan(p); return rc; }
    *out = p;
    return PP_SUCCESS;
}

int pp_solve(const pp_plan *plan, const double *f, double *u, void *stream) {
    if (!plan || !f || !u) return PP_ERR_NULL;
    const size_t n = (size_t)plan->nx * plan->ny * plan->nz;
    if (((uintptr_t)f & 15) || ((uintptr_t)u & 15)) return PP_ERR_INVALID_ARG;
    if (f != u) {
        const uintptr_t a = (uintptr_t)f, b = (uintptr_t)u, len = n * sizeof(double);
        if (a < b + len && b < a + len) return PP_ERR_INVALID_ARG;     // partial overlap
    }
    cudaStream_t st = (cudaStream_t)stream;
    pp_plan *mp = const_cast<pp_plan *>(plan);
    const bool prof = plan->profiling != 0;
    int rc;
#define PP_MARK(i) if (prof && cudaEventRecord(mp->ev[i], st) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    const bool fused = plan->xy_fusion && fusion_supported(plan->nx, plan->ny);
    PP_MARK(0)
    if (fused) {
        if ((rc = run_fused(plan, true, f, u, st))) return rc;  // a1-a6 as tasks of one kernel
        PP_MARK(1)
    } else {
        if ((rc = run_x(plan, true, f, u, st))) return rc;      // a1-a3: x pre / FFT / post
        PP_MARK(1)
        if ((rc = run_y(plan, true, u, st))) return rc;         // a4-a6: y pre / FFT / post
    }
    PP_MARK(2)
    if ((rc = run_z(plan, u, st))) return rc;                   // a7-a8: diagonal + tridiagonal solve
    PP_MARK(3)
    if (fused) {
        PP_MARK(4)
        if ((rc = run_fused(plan, false, u, u, st))) return rc; // a9-a10 as tasks of one kernel
    } else {
        if ((rc = run_y(plan, false, u, st))) return rc;        // a9: y inverse
        PP_MARK(4)
        if ((rc = run_x(plan, false, u, u, st))) return rc;     // a10: x inverse
    }
    PP_MARK(5)
#undef PP_MARK
    if (prof) mp->have_times = 1;
    return PP_SUCCESS;
}

int pp_solve_host(pp_plan *plan, const double *f_host, double *u_host, void *stream) {
    if (!plan || !f_host || !u_host) return PP_ERR_NULL;
    const size_t nb = (size_t)plan->nx * plan->ny * plan->nz * sizeof(double);
    if (!plan->host_stage) {
        if (cudaMalloc((void **)&plan->host_stage, nb) != cudaSuccess) {
            plan->host_stage = nullptr;
            cudaGetLastError();
            return PP_ERR_ALLOC;
        }
        plan->bytes += nb;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMemcpyAsync(plan->host_stage, f_host, nb, cudaMemcpyHostToDevice, st) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    if (int rc = pp_solve(plan, plan->host_stage, plan->host_stage, stream)) return rc;
    if (cudaMemcpyAsync(u_host, plan->host_stage, nb, cudaMemcpyDeviceToHost, st) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    if (cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    return PP_SUCCESS;
}

int pp_solve_host_batch(pp_plan *plan, const double *f_host, double *u_host, int nbatch, void *stream) {
    if (!plan || !f_host || !u_host) return PP_ERR_NULL;
    if (nbatch < 1) return PP_ERR_INVALID_ARG;
    const size_t n = (size_t)plan->nx * plan->ny * plan->nz, nb = n * sizeof(double);
    cudaStream_t st = (cudaStream_t)stream;
    const int nstage = nbatch < pp_plan::NSTAGE ? nbatch : pp_plan::NSTAGE;
    // lazily: staging ring, copy streams, events
    if (!plan->s_in) {
        if (cudaStreamCreateWithFlags(&plan->s_in, cudaStreamNonBlocking) != cudaSuccess ||
            cudaStreamCreateWithFlags(&plan->s_out, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    }
    for (int b = 0; b < nstage; ++b) {
        if (!plan->batch_stage[b]) {
            if (cudaMalloc((void **)&plan->batch_stage[b], nb) != cudaSuccess) { plan->batch_stage[b] = nullptr; cudaGetLastError(); return PP_ERR_ALLOC; }
            plan->bytes += nb;
        }
        if (!plan->ev_in[b]) {
            if (cudaEventCreateWithFlags(&plan->ev_in[b], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&plan->ev_done[b], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&plan->ev_out[b], cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
        }
    }
#define PP_CK(call) if ((call) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    // copy-in of right-hand side i+1 and copy-out of solution i-1 run beside the solve of i (PCIe is full duplex)
    for (int i = 0; i < nbatch; ++i) {
        const int b = i % nstage;
        double *d = plan->batch_stage[b];
        if (i >= nstage) PP_CK(cudaStreamWaitEvent(plan->s_in, plan->ev_out[b], 0))          // buffer free again
        PP_CK(cudaMemcpyAsync(d, f_host + (size_t)i * n, nb, cudaMemcpyHostToDevice, plan->s_in))
        PP_CK(cudaEventRecord(plan->ev_in[b], plan->s_in))
        PP_CK(cudaStreamWaitEvent(st, plan->ev_in[b], 0))
        if (int rc = pp_solve(plan, d, d, stream)) return rc;
        PP_CK(cudaEventRecord(plan->ev_done[b], st))
        PP_CK(cudaStreamWaitEvent(plan->s_out, plan->ev_done[b], 0))
        PP_CK(cudaMemcpyAsync(u_host + (size_t)i * n, d, nb, cudaMemcpyDeviceToHost, plan->s_out))
        PP_CK(cudaEventRecord(plan->ev_out[b], plan->s_out))
    }
    PP_CK(cudaStreamSynchronize(plan->s_out))
    PP_CK(cudaStreamSynchronize(st))
#undef PP_CK
    return PP_SUCCESS;
}

int pp_plan_destroy(pp_plan *plan) {
    free_plan(plan);
    return PP_SUCCESS;
}

size_t pp_plan_workspace_bytes(const pp_plan *plan) { return plan ? plan->bytes : 0; }

int pp_plan_set_profiling(pp_plan *plan, int enable) {
    if (!plan) return PP_ERR_NULL;
    plan->profiling = enable ? 1 : 0;
    plan->have_times = 0;
    return PP_SUCCESS;
}

int pp_plan_set_z_algorithm(pp_plan *plan, int algorithm) {
    if (!plan) return PP_ERR_NULL;
    if (algorithm != PP_Z_AUTO && algorithm != PP_Z_SWEEP && algorithm != PP_Z_PARTITION) return PP_ERR_INVALID_ARG;
    if (algorithm == PP_Z_PARTITION && plan_zpart_shape(plan).R == 0 && !plan->hier_scratch)
        return PP_ERR_UNSUPPORTED_SIZE;
    if (algorithm == PP_Z_SWEEP && plan->nz > 64 * Z_MAX_CK) return PP_ERR_UNSUPPORTED_SIZE;
    plan->z_algorithm = algorithm;
    return PP_SUCCESS;
}

int pp_plan_set_xy_fusion(pp_plan *plan, int enable) {
    if (!plan) return PP_ERR_NULL;
    if (enable && !fusion_supported(plan->nx, plan->ny)) return PP_ERR_UNSUPPORTED_SIZE;
    plan->xy_fusion = enable ? 1 : 0;
    return PP_SUCCESS;
}

int pp_fold_dirichlet(const pp_plan *plan, double *f, const double *gx_lo, const double *gx_hi, const double *gy_lo,
                      const double *gy_hi, const double *gz_lo, const double *gz_hi, void *stream) {
    if (!plan || !f) return PP_ERR_NULL;
    if (((gx_lo || gx_hi) && plan->bcx != PP_BC_DIRICHLET) || ((gy_lo || gy_hi) && plan->bcy != PP_BC_DIRICHLET) ||
        ((gz_lo || gz_hi) && plan->bcz != PP_BC_DIRICHLET))
        return PP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const long long nx = plan->nx, ny = plan->ny, nz = plan->nz;
    auto fold = [&](const double *g, long long nf, long long ns, long long sf, long long ss, long long offset, double h) {
        if (!g) return;
        const dim3 grid((unsigned)((nf + 127) / 128), (unsigned)ns);
        fold_face_kernel<<<grid, 128, 0, st>>>(f, g, (int)nf, (int)ns, sf, ss, offset, 2.0 / (h * h));
    };
    fold(gx_lo, ny, nz, nx, nx * ny, 0, plan->dx);                        // g[k][j] -> cell (0, j, k)
    fold(gx_hi, ny, nz, nx, nx * ny, nx - 1, plan->dx);
    fold(gy_lo, nx, nz, 1, nx * ny, 0, plan->dy);                         // g[k][i] -> cell (i, 0, k)
    fold(gy_hi, nx, nz, 1, nx * ny, (ny - 1) * nx, plan->dy);
    fold(gz_lo, nx, ny, 1, nx, 0, plan->dz);                              // g[j][i] -> cell (i, j, 0)
    fold(gz_hi, nx, ny, 1, nx, (nz - 1) * nx * ny, plan->dz);
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}

int pp_plan_set_null_space(pp_plan *plan, int convention) {
    if (!plan) return PP_ERR_NULL;
    if (convention != PP_NULL_ZERO_MEAN && convention != PP_NULL_PIN_PLANE0) return PP_ERR_INVALID_ARG;
    plan->null_space = convention;
    return PP_SUCCESS;
}

int pp_size_supported(int nx, int ny, int nz, int bc_z) {
    if (bc_z != PP_BC_PERIODIC && bc_z != PP_BC_NEUMANN && bc_z != PP_BC_DIRICHLET) return 0;
    const bool long_ok = bc_z != PP_BC_PERIODIC && zpart_hier_ok(nz);
    return (length_supported(nx) && length_supported(ny) && nz >= 2 && (nz <= 64 * Z_MAX_CK || long_ok)) ? 1 : 0;
}

int pp_plan_launches_per_solve(const pp_plan *plan) {
    if (!plan) return 0;
    const bool fused = plan->xy_fusion && fusion_supported(plan->nx, plan->ny);
    int n = fused ? 2 : 4;                                        // x/y passes
    const bool want_part = plan->z_algorithm != PP_Z_SWEEP;
    if (want_part && plan_zpart_shape(plan).R == 0 && plan->hier_scratch) n += 3 + (plan->singular ? 1 : 0);
    else n += 1;
    return n;
}

int pp_plan_last_kernel_ms(pp_plan *plan, float *ms_out) {
    if (!plan || !ms_out) return PP_ERR_NULL;
    if (!plan->have_times) return PP_ERR_INVALID_ARG;
    if (cudaEventSynchronize(plan->ev[PP_NUM_KERNELS]) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    for (int i = 0; i < PP_NUM_KERNELS; ++i)
        if (cudaEventElapsedTime(&ms_out[i], plan->ev[i], plan->ev[i + 1]) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    return PP_SUCCESS;
}

}  // extern "C"
