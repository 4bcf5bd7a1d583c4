// C ABI of pittpack_b200 (include/pittpack_b200.h): plan construction, table generation and the
// five-kernel solve.  No cuFFT / cuSPARSE, no CPU fallback.

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "pp_plan.h"
#include "pp_xpass.cuh"      // XCfg: the radix schedule of the x pass (twiddle tables)
#include "pp_ypass.cuh"      // YCfg, YRows
#include "pp_zshape.h"       // zpart_shape, zpart_hier_ok, Z_MAX_CK (host-side size rules)

using namespace pp;

namespace pp {
// largest dynamic shared-memory size each (device, kernel) has been opted in to: the attribute is only ever raised
static std::mutex g_smem_mutex;
static std::map<std::pair<int, const void *>, size_t> g_smem_max;

int set_smem_once(const void *kernel, size_t smem) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(g_smem_mutex);
    size_t &have = g_smem_max[std::make_pair(dev, kernel)];
    if (smem <= have) return PP_SUCCESS;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        cudaGetLastError();
        return PP_ERR_CUDA;
    }
    have = smem;
    return PP_SUCCESS;
}
}  // namespace pp

// ------------------------------------------------------------------------------------------
// host-side tables, evaluated in long double and rounded once
// ------------------------------------------------------------------------------------------
namespace {

const long double PI_L = 3.14159265358979323846264338327950288L;

constexpr int PP_MAX_NZ = 16384;        // longest z line (the paper's pencils)

// powers of two in [4, 2048], 3 * 2^k in [48, 1536], 5 * 2^k in [80, 1280]
bool length_supported(int n) { return n >= 4 && n <= 2048 && fft_length_ok(n); }

// e: elements per thread of the pass that will use the table (fixes the radix schedule, pp_fft.cuh)
void make_twiddles(int n, int e, std::vector<double2> &tw, std::vector<double2> &ptw) {
    tw.assign(tw_table_elems(n, e), make_double2(1.0, 0.0));
    ptw.resize(n + 1);
    // stage with NS: row r = 1 (radix 8, 16) or rows r = 1, 2 (radix 4) of W_n^(k r stride), stride = n / (RS NS), k in [0, NS)
    const int rs = stage_radix(n, e), rows = tw_rows(n, e);
    for (int ns = first_radix(n, e); ns < n; ns *= rs) {
        const int off = tw_stage_offset(n, e, ns), stride = n / (rs * ns);
        for (int ri = 0; ri < rows; ++ri)
            for (int k = 0; k < ns; ++k) {
                const long long ex = ((long long)k * (1 << ri) * stride) % n;
                const long double a = 2.0L * PI_L * (long double)ex / (long double)n;
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

void free_plan(pp_plan *p) {
    if (!p) return;
    if (p->tw_xi != p->tw_x) cudaFree(p->tw_xi);
    cudaFree(p->tw_x); cudaFree(p->tw_y); cudaFree(p->ptw_x); cudaFree(p->ptw_y);
    cudaFree(p->sx); cudaFree(p->sy); cudaFree(p->zero_scratch); cudaFree(p->host_stage); cudaFree(p->fuse_sync); cudaFree(p->hier_scratch);
    for (auto &e : p->ev) if (e) cudaEventDestroy(e);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->side) cudaStreamDestroy(p->side);
    for (auto &e : p->ev_pipe) if (e) cudaEventDestroy(e);
    if (p->ev_pipe_join) cudaEventDestroy(p->ev_pipe_join);
    if (p->pipe) cudaStreamDestroy(p->pipe);
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
        case PP_ERR_UNSUPPORTED_SIZE: return "unsupported grid size (nx, ny: 2^k in [4, 2048], 3*2^k in [48, 1536] or 5*2^k in [80, 1280]; nz in [2, 16384])";
        case PP_ERR_ALLOC: return "allocation failed";
        case PP_ERR_CUDA: return "CUDA runtime or launch error (is a CUDA device present?)";
        case PP_ERR_NULL: return "null pointer argument";
        case PP_ERR_STATIC_LIMIT: return "nz is beyond PP_STATIC_MAX_NZ = 4096, the fixed work line of pp_zsolve_static (longer lines need a plan)";
        default: return "unknown status";
    }
}

// ny_z: the number of ky rows the z solve of this plan will see -- ny, or ny / world for the z-side plan of a slab
// decomposition (its kernel choice and its two-level scratch follow the pencil, not the whole plane)
static int plan_create_impl(pp_plan **out, int nx, int ny, int nz, double dx, double dy, double dz,
                            int bc_x, int bc_y, int bc_z, int ny_z);

int pp_plan_create(pp_plan **out, int nx, int ny, int nz, double dx, double dy, double dz,
                   int bc_x, int bc_y, int bc_z) {
    return plan_create_impl(out, nx, ny, nz, dx, dy, dz, bc_x, bc_y, bc_z, ny);
}

}  // extern "C"

static int plan_create_impl(pp_plan **out, int nx, int ny, int nz, double dx, double dy, double dz,
                            int bc_x, int bc_y, int bc_z, int ny_z) {
    if (!out) return PP_ERR_NULL;
    *out = nullptr;
    if (nx <= 0 || ny <= 0 || nz <= 0) return PP_ERR_INVALID_ARG;
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz))
        return PP_ERR_INVALID_ARG;
    for (int bc : {bc_x, bc_y, bc_z})
        if (bc != PP_BC_PERIODIC && bc != PP_BC_NEUMANN && bc != PP_BC_DIRICHLET) return PP_ERR_INVALID_ARG;
    // nz: any value in [2, 16384].  Multiples of 256 beyond what one CTA holds go to the two-level partition,
    // everything the partitioned kernels do not take to the two-sweep kernels.
    const bool long_ok = zpart_hier_ok(nz);
    if (!length_supported(nx) || !length_supported(ny) || nz < 2 || nz > PP_MAX_NZ) return PP_ERR_UNSUPPORTED_SIZE;

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
    make_twiddles(nx, fft_E(nx, PP_X_E16_MIN), tw, ptw);
    if (!rc) rc = upload(&p->tw_x, tw, p->bytes);
    if (!rc) rc = upload(&p->ptw_x, ptw, p->bytes);
    p->tw_xi = p->tw_x;
    if (fft_E(nx, PP_XI_E16_MIN) != fft_E(nx, PP_X_E16_MIN)) {      // the inverse x pass runs another radix schedule
        p->tw_xi = nullptr;
        make_twiddles(nx, fft_E(nx, PP_XI_E16_MIN), tw, ptw);
        if (!rc) rc = upload(&p->tw_xi, tw, p->bytes);
    }
    make_twiddles(ny, fft_E(ny, PP_Y_E16_MIN), tw, ptw);
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
    if (!rc) {
        std::vector<double> z((size_t)nz * Z_MAX_BATCH, 0.0);
        rc = upload(&p->zero_scratch, z, p->bytes);
    }
    // two-level partition (segments of 32 rows; its interface kernels carry the minors over up to 33 rows between
    // renormalisations, hence the range check): interface values [2][nK][plane] + scratch [2][nK][plane], or
    // [6][nK][plane] when the chain of super-segments is cyclic (periodic z)
    p->ny = ny_z;                                  // (the cluster rule looks at the number of lines the z solve sees)
    const bool z_cluster = zpart_cluster(p);
    p->ny = ny;
    if (!rc && long_ok && zpart_shape(nz).R == 0 && zpart_range_ok(p, 33) && !z_cluster) {
        const size_t nb = sizeof(double) * (bc_z == PP_BC_PERIODIC ? 8 : 4) * (size_t)(nz / ZP_HIER_ROWS) * (size_t)nx * (size_t)ny_z;
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

extern "C" {

// a plan's tables live on the device that was current at pp_plan_create: every call that launches must
// find the same device current (a status code instead of an illegal-address fault at the next sync)
static int check_device(const pp_plan *plan) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    return dev == plan->device ? PP_SUCCESS : PP_ERR_INVALID_ARG;
}

int pp_solve(const pp_plan *plan, const double *f, double *u, void *stream) {
    if (!plan || !f || !u) return PP_ERR_NULL;
    if (int rc = check_device(plan)) return rc;
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
    // x/y slab pipeline: pass A of slab k on the caller's stream, pass B of slab k on the plan's second stream as soon
    // as A(k) is done -- beside A(k+1); the caller's stream joins at the end
    const int pipe = (plan->xy_pipeline > 0 && plan->xy_pipeline < plan->nz && !fused) ? plan->xy_pipeline : 0;
    auto pipelined = [&](bool fwd) -> int {
        const int nslab = (plan->nz + pipe - 1) / pipe;
        for (int k = 0; k < nslab; ++k) {
            const int z0 = k * pipe, nzs = (plan->nz - z0 < pipe) ? plan->nz - z0 : pipe;
            int r = fwd ? run_x(plan, true, f, u, st, z0, nzs) : run_y_inv(plan, u, nullptr, st, z0, nzs);
            if (r) return r;
            if (cudaEventRecord(mp->ev_pipe[k], st) != cudaSuccess || cudaStreamWaitEvent(mp->pipe, mp->ev_pipe[k], 0) != cudaSuccess) {
                cudaGetLastError();
                return PP_ERR_CUDA;
            }
            r = fwd ? run_y_fwd(plan, u, nullptr, mp->pipe, z0, nzs) : run_x(plan, false, u, u, mp->pipe, z0, nzs);
            if (r) return r;
        }
        if (cudaEventRecord(mp->ev_pipe_join, mp->pipe) != cudaSuccess || cudaStreamWaitEvent(st, mp->ev_pipe_join, 0) != cudaSuccess) {
            cudaGetLastError();
            return PP_ERR_CUDA;
        }
        return PP_SUCCESS;
    };
    PP_MARK(0)
    if (pipe) {
        if ((rc = pipelined(true))) return rc;
        PP_MARK(1)
    } else if (fused) {
        if ((rc = run_fused(plan, true, f, u, st))) return rc;  // a1-a6 as tasks of one kernel
        PP_MARK(1)
    } else {
        if ((rc = run_x(plan, true, f, u, st))) return rc;      // a1-a3: x pre / FFT / post
        PP_MARK(1)
        if ((rc = run_y_fwd(plan, u, nullptr, st))) return rc;         // a4-a6: y pre / FFT / post
    }
    PP_MARK(2)
    if ((rc = run_z(plan, u, st))) return rc;                   // a7-a8: diagonal + tridiagonal solve
    PP_MARK(3)
    if (pipe) {
        PP_MARK(4)
        if ((rc = pipelined(false))) return rc;
    } else if (fused) {
        PP_MARK(4)
        if ((rc = run_fused(plan, false, u, u, st))) return rc; // a9-a10 as tasks of one kernel
    } else {
        if ((rc = run_y_inv(plan, u, nullptr, st))) return rc;        // a9: y inverse
        PP_MARK(4)
        if ((rc = run_x(plan, false, u, u, st))) return rc;     // a10: x inverse
    }
    PP_MARK(5)
#undef PP_MARK
    if (prof) mp->have_times = 1;
    return PP_SUCCESS;
}

int pp_solve_batch(const pp_plan *plan, const double *f, double *u, int nbatch, void *stream) {
    if (!plan || !f || !u) return PP_ERR_NULL;
    if (nbatch < 1) return PP_ERR_INVALID_ARG;
    if (int rc = check_device(plan)) return rc;
    const size_t n = (size_t)plan->nx * plan->ny * plan->nz;
    if ((long long)plan->nz * nbatch > 0x7fffffffLL) return PP_ERR_INVALID_ARG;
    if (((uintptr_t)f & 15) || ((uintptr_t)u & 15)) return PP_ERR_INVALID_ARG;
    if (f != u) {
        const uintptr_t a = (uintptr_t)f, b = (uintptr_t)u, len = n * nbatch * sizeof(double);
        if (a < b + len && b < a + len) return PP_ERR_INVALID_ARG;     // partial overlap
    }
    cudaStream_t st = (cudaStream_t)stream;
    // the y passes put one plane per blockIdx.y, and a grid's y extent ends at 65535: the stack is cut into groups of
    // at most floor(65535 / nz) grids (>= 3, nz <= 16384), each group one launch per transform pass
    const int group = 65535 / plan->nz;
    for (int i0 = 0; i0 < nbatch; i0 += group) {
        const int nb = (nbatch - i0 < group) ? nbatch - i0 : group;
        const int planes = plan->nz * nb;
        const double *fg = f + (size_t)i0 * n;
        double *ug = u + (size_t)i0 * n;
        int rc;
        if ((rc = run_x(plan, true, fg, ug, st, 0, planes))) return rc;        // a1-a3 of every right-hand side of the group
        if ((rc = run_y_fwd(plan, ug, nullptr, st, 0, planes))) return rc;     // a4-a6
        if ((rc = run_z(plan, ug, st, nb))) return rc;                         // a7-a8 (up to 64 grids per launch where one CTA holds a line)
        if ((rc = run_y_inv(plan, ug, nullptr, st, 0, planes))) return rc;     // a9
        if ((rc = run_x(plan, false, ug, ug, st, 0, planes))) return rc;       // a10
    }
    return PP_SUCCESS;
}

int pp_solve_host(pp_plan *plan, const double *f_host, double *u_host, void *stream) {
    if (!plan || !f_host || !u_host) return PP_ERR_NULL;
    if (int rc = check_device(plan)) return rc;
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
    if (int rc = check_device(plan)) return rc;
    const size_t n = (size_t)plan->nx * plan->ny * plan->nz, nb = n * sizeof(double);
    cudaStream_t st = (cudaStream_t)stream;
    const int nstage = nbatch < pp_plan::NSTAGE ? nbatch : pp_plan::NSTAGE;
    // lazily: staging ring, copy streams, events
    // (each handle is tested on its own, so a creation that failed half-way is completed by the next call instead of
    // leaving a NULL stream or event in use)
    for (cudaStream_t *s : {&plan->s_in, &plan->s_out})
        if (!*s && cudaStreamCreateWithFlags(s, cudaStreamNonBlocking) != cudaSuccess) { *s = nullptr; cudaGetLastError(); return PP_ERR_CUDA; }
    for (int b = 0; b < nstage; ++b) {
        if (!plan->batch_stage[b]) {
            if (cudaMalloc((void **)&plan->batch_stage[b], nb) != cudaSuccess) { plan->batch_stage[b] = nullptr; cudaGetLastError(); return PP_ERR_ALLOC; }
            plan->bytes += nb;
        }
        for (cudaEvent_t *e : {&plan->ev_in[b], &plan->ev_done[b], &plan->ev_out[b]})
            if (!*e && cudaEventCreateWithFlags(e, cudaEventDisableTiming) != cudaSuccess) { *e = nullptr; cudaGetLastError(); return PP_ERR_CUDA; }
    }
    // on an error in mid-batch the copies and solves already enqueued still use the staging ring: wait for
    // them before returning, so that a later call cannot reuse a buffer that is in flight
    auto drain = [&](int rc) {
        cudaStreamSynchronize(plan->s_in);
        cudaStreamSynchronize(plan->s_out);
        cudaStreamSynchronize(st);
        cudaGetLastError();
        return rc;
    };
#define PP_CK(call) if ((call) != cudaSuccess) { cudaGetLastError(); return drain(PP_ERR_CUDA); }
    // copy-in of right-hand side i+1 and copy-out of solution i-1 run beside the solve of i (PCIe is full duplex)
    for (int i = 0; i < nbatch; ++i) {
        const int b = i % nstage;
        double *d = plan->batch_stage[b];
        if (i >= nstage) PP_CK(cudaStreamWaitEvent(plan->s_in, plan->ev_out[b], 0))          // buffer free again
        PP_CK(cudaMemcpyAsync(d, f_host + (size_t)i * n, nb, cudaMemcpyHostToDevice, plan->s_in))
        PP_CK(cudaEventRecord(plan->ev_in[b], plan->s_in))
        PP_CK(cudaStreamWaitEvent(st, plan->ev_in[b], 0))
        if (int rc = pp_solve(plan, d, d, stream)) return drain(rc);
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

// ---- slab decomposition (include/pittpack_b200.h, "Slab decomposition") --------------------------------------
struct pp_slab_plan {
    int world, rank;
    pp_plan *slab;      // nx x ny x nz/world: tables of the x and y passes
    pp_plan *full;      // nx x ny x nz: z-solve tables (shift tables, scratch); never solved as a whole
    pp_plan zview;      // `full` seen from this rank's pencil: ny/world rows starting at ky = rank ny/world
    YRows fwd, inv;
    int have_exchange;
};

int pp_slab_plan_create(pp_slab_plan **out, int world, int rank, int nx, int ny, int nz, double dx, double dy, double dz,
                        int bc_x, int bc_y, int bc_z) {
    if (!out) return PP_ERR_NULL;
    *out = nullptr;
    if (world < 1 || world > PP_MAX_WORLD || rank < 0 || rank >= world) return PP_ERR_INVALID_ARG;
    if (nz <= 0 || ny <= 0 || nz % world || ny % world || nz / world < 2) return PP_ERR_UNSUPPORTED_SIZE;
    pp_slab_plan *sp = new (std::nothrow) pp_slab_plan();
    if (!sp) return PP_ERR_ALLOC;
    std::memset(sp, 0, sizeof(*sp));
    sp->world = world; sp->rank = rank;
    int rc = pp_plan_create(&sp->slab, nx, ny, nz / world, dx, dy, dz, bc_x, bc_y, bc_z);
    if (!rc) rc = plan_create_impl(&sp->full, nx, ny, nz, dx, dy, dz, bc_x, bc_y, bc_z, ny / world);
    if (rc) { free_plan(sp->slab); free_plan(sp->full); delete sp; return rc; }
    const int nyl = ny / world;
    sp->zview = *sp->full;                       // shares full's device tables; owns nothing
    sp->zview.ny = nyl;
    sp->zview.sy = sp->full->sy + (size_t)rank * nyl;
    sp->zview.singular = (sp->full->singular && rank == 0) ? 1 : 0;     // the (0,0) mode is element 0 of rank 0's pencil
    sp->fwd.rpb = sp->inv.rpb = nyl;
    *out = sp;
    return PP_SUCCESS;
}

int pp_slab_plan_destroy(pp_slab_plan *plan) {
    if (!plan) return PP_SUCCESS;
    free_plan(plan->slab);
    free_plan(plan->full);
    delete plan;
    return PP_SUCCESS;
}

size_t pp_slab_local_elems(const pp_slab_plan *plan) {
    return plan ? (size_t)plan->full->nx * plan->full->ny * plan->full->nz / plan->world : 0;
}
size_t pp_slab_chunk_elems(const pp_slab_plan *plan) { return plan ? pp_slab_local_elems(plan) / plan->world : 0; }

int pp_slab_set_exchange(pp_slab_plan *plan, double *const *fwd_dst, const double *const *inv_src) {
    if (!plan || !fwd_dst || !inv_src) return PP_ERR_NULL;
    for (int q = 0; q < plan->world; ++q) {
        if (!fwd_dst[q] || !inv_src[q]) return PP_ERR_NULL;
        if (((uintptr_t)fwd_dst[q] & 15) || ((uintptr_t)inv_src[q] & 15)) return PP_ERR_INVALID_ARG;
        plan->fwd.base[q] = (double2 *)fwd_dst[q];
        plan->inv.base[q] = (double2 *)const_cast<double *>(inv_src[q]);
    }
    plan->have_exchange = 1;
    return PP_SUCCESS;
}

int pp_slab_forward(const pp_slab_plan *plan, const double *f_slab, double *work_slab, void *stream) {
    if (!plan || !f_slab || !work_slab) return PP_ERR_NULL;
    if (!plan->have_exchange) return PP_ERR_INVALID_ARG;
    if (((uintptr_t)f_slab & 15) || ((uintptr_t)work_slab & 15)) return PP_ERR_INVALID_ARG;
    if (int rc = check_device(plan->slab)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (int rc = run_x(plan->slab, true, f_slab, work_slab, st)) return rc;       // a1-a3 on the slab
    return run_y_fwd(plan->slab, work_slab, &plan->fwd, st);                // a4-a6, rows stored to their owners
}

int pp_slab_zsolve(const pp_slab_plan *plan, double *pencil, void *stream) {
    if (!plan || !pencil) return PP_ERR_NULL;
    if ((uintptr_t)pencil & 15) return PP_ERR_INVALID_ARG;
    if (int rc = check_device(plan->full)) return rc;
    return run_z(&plan->zview, pencil, (cudaStream_t)stream);                     // a7-a8 on nx * ny/world systems
}

int pp_slab_inverse(const pp_slab_plan *plan, double *u_slab, void *stream) {
    if (!plan || !u_slab) return PP_ERR_NULL;
    if (!plan->have_exchange) return PP_ERR_INVALID_ARG;
    if ((uintptr_t)u_slab & 15) return PP_ERR_INVALID_ARG;
    if (int rc = check_device(plan->slab)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (int rc = run_y_inv(plan->slab, u_slab, &plan->inv, st)) return rc; // a9, rows loaded from their owners
    return run_x(plan->slab, false, u_slab, u_slab, st);                          // a10
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
    if (algorithm != PP_Z_AUTO && algorithm != PP_Z_SWEEP && algorithm != PP_Z_PARTITION && algorithm != PP_Z_CLUSTER) return PP_ERR_INVALID_ARG;
    if (algorithm == PP_Z_CLUSTER && !zpart_cluster_possible(plan)) return PP_ERR_UNSUPPORTED_SIZE;
    if (algorithm == PP_Z_PARTITION && !zpart_single_level(plan) && !plan->hier_scratch)
        return PP_ERR_UNSUPPORTED_SIZE;
    plan->z_algorithm = algorithm;
    return PP_SUCCESS;
}

int pp_plan_set_xy_pipeline(pp_plan *plan, int planes_per_slab) {
    if (!plan) return PP_ERR_NULL;
    if (planes_per_slab < 0) return PP_ERR_INVALID_ARG;
    if (int rc = check_device(plan)) return rc;
    if (planes_per_slab > 0) {
        if ((plan->nz + planes_per_slab - 1) / planes_per_slab > pp_plan::MAX_PIPE) return PP_ERR_INVALID_ARG;
        // each handle tested on its own: a creation that failed half-way is completed by the next call, and the
        // pipeline is only switched on (below) once every stream and event exists
        if (!plan->pipe && cudaStreamCreateWithFlags(&plan->pipe, cudaStreamNonBlocking) != cudaSuccess) { plan->pipe = nullptr; cudaGetLastError(); return PP_ERR_CUDA; }
        for (auto &e : plan->ev_pipe)
            if (!e && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { e = nullptr; cudaGetLastError(); return PP_ERR_CUDA; }
        if (!plan->ev_pipe_join && cudaEventCreateWithFlags(&plan->ev_pipe_join, cudaEventDisableTiming) != cudaSuccess) { plan->ev_pipe_join = nullptr; cudaGetLastError(); return PP_ERR_CUDA; }
    }
    plan->xy_pipeline = planes_per_slab;
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
    if (int rc = check_device(plan)) return rc;
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
    return (length_supported(nx) && length_supported(ny) && nz >= 2 && nz <= PP_MAX_NZ) ? 1 : 0;
}

int pp_plan_launches_per_solve(const pp_plan *plan) {
    if (!plan) return 0;
    const bool fused = plan->xy_fusion && fusion_supported(plan->nx, plan->ny);
    int n = fused ? 2 : 4;                                        // x/y passes
    if (!fused && plan->xy_pipeline > 0 && plan->xy_pipeline < plan->nz)
        n = 4 * ((plan->nz + plan->xy_pipeline - 1) / plan->xy_pipeline);       // ... slab by slab
    const bool want_part = plan->z_algorithm != PP_Z_SWEEP;
    if (want_part && zpart_cluster(plan)) n += 1 + (plan->singular ? 1 : 0);
    else if (want_part && !zpart_single_level(plan) && plan->hier_scratch) n += 3 + (plan->singular ? 1 : 0);
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
