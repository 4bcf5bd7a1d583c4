// z-solve launcher (a7-a8): picks the partitioned, two-level or two-sweep kernels.
#include <climits>
#include <cmath>
#include <cstdint>
#include <mutex>

#include "pp_plan.h"
#include "pp_zsolve.cuh"
#include "pp_zpart.cuh"

namespace pp {

// The partitioned z kernels tabulate the leading minors q_0 .. q_R of a segment block, |q_R| <= bmax^R:
// for grids so anisotropic (dz >> dx) that this could leave the fp64 range they are not used.
bool zpart_range_ok(const pp_plan *p, int R) { return (double)R * std::log2(p->bmax) < 1000.0; }
static ZPartShape plan_zpart_shape(const pp_plan *p) {
    const ZPartShape z = zpart_shape(p->nz);
    return (z.R && zpart_range_ok(p, z.R)) ? z : ZPartShape{0, 0, 0};
}

bool zpart_cluster_possible(const pp_plan *p) { return zpart_cluster_possible(p->nz, p->bcz == PP_BC_PERIODIC) && zpart_range_ok(p, 33); }
bool zpart_cluster(const pp_plan *p) {
    if (p->z_algorithm == PP_Z_CLUSTER) return zpart_cluster_possible(p);
    return zpart_cluster_ok(p->nz, (long long)p->nx * p->ny, p->bcz == PP_BC_PERIODIC) && zpart_range_ok(p, 33);
}
bool zpart_single_level(const pp_plan *p) { return zpart_cluster(p) || plan_zpart_shape(p).R != 0; }

static int run_z_one(const pp_plan *p, double *w, cudaStream_t st, int nbatch);

int run_z(const pp_plan *p, double *w, cudaStream_t st, int nbatch) {
    const size_t n = (size_t)p->nx * p->ny * p->nz;
    // the one-CTA partitioned kernel takes up to Z_MAX_BATCH grids per launch (blockIdx.y); every other kernel one
    const bool batched = p->z_algorithm != PP_Z_SWEEP && !zpart_cluster(p) && plan_zpart_shape(p).R != 0;
    const int step = batched ? Z_MAX_BATCH : 1;
    for (int i = 0; i < nbatch; i += step)
        if (int rc = run_z_one(p, w + (size_t)i * n, st, (nbatch - i < step) ? nbatch - i : step)) return rc;
    return PP_SUCCESS;
}

static int run_z_one(const pp_plan *p, double *w, cudaStream_t st, int nbatch) {
    ZParams zp;
    zp.batch_stride = (size_t)p->nx * p->ny * p->nz;
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
    if (want_part && zpart_cluster(p)) {
        // two levels in one pass: a cluster of nz / 256 CTAs per line, super-segment interfaces through distributed
        // shared memory (pp_zpart.cuh, MODE 3): one HBM read + one write per unknown
        const ZPartShape hs = {32, ZP_HIER_ROWS / 32, 32};
        const size_t ds = zpart_smem_bytes(hs, false, true);
        const int nK = p->nz / ZP_HIER_ROWS;
        const ZHier h = {nK, nullptr, nullptr, 0};
        auto kernel = zsolve_part_kernel<32, 3, false>;
        if (int rc = set_smem(kernel, ds)) return rc;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)((plane + hs.L - 1) / hs.L), (unsigned)nK);
        cfg.blockDim = dim3((unsigned)(hs.L * hs.S));
        cfg.dynamicSmemBytes = ds;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 1;
        attr[0].val.clusterDim.y = (unsigned)nK;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (cudaLaunchKernelEx(&cfg, kernel, w, zp, hs.S, hs.L, h) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
        // the singular (0,0) line: column 0 only, which the cluster kernel reads but never stores
        if (p->singular)
            zero_mode_long_kernel<<<1, 1024, 0, st>>>(w, plane, p->nz, p->scale, p->null_space == PP_NULL_PIN_PLANE0, 0);
    } else if (zs.R) {
        // partitioned, register-resident solve: one HBM read + one write per unknown (pp_zpart.cuh)
        const bool cyc = p->bcz == PP_BC_PERIODIC;
        const size_t ds = zpart_smem_bytes(zs, cyc);
        const dim3 grid((unsigned)((plane + zs.L - 1) / zs.L), (unsigned)nbatch);
        const ZHier none = {1, nullptr, nullptr, 0};
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
        const bool per = p->bcz == PP_BC_PERIODIC;
        const ZHier h = {nK, p->hier_scratch, p->hier_scratch + slab, per ? 1 : 0};
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
            zero_mode_long_kernel<<<1, 1024, 0, p->side>>>(w, plane, p->nz, p->scale, p->null_space == PP_NULL_PIN_PLANE0, per ? 1 : 0);
            if (cudaEventRecord(p->ev_join, p->side) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
        }
        zsolve_part_kernel<32, 1><<<grid, hs.L * hs.S, ds, st>>>(w, zp, hs.S, hs.L, h);
        if (per)
            zsolve_hier_interface_cyclic_kernel<<<(unsigned)((plane + 63) / 64), 64, 0, st>>>(zp, h, ZP_HIER_ROWS, p->hier_scratch + 2 * slab);
        else
            zsolve_hier_interface_kernel<<<(unsigned)((plane + 63) / 64), 64, 0, st>>>(zp, h, ZP_HIER_ROWS, p->hier_scratch + 2 * slab,
                                                                                 p->hier_scratch + 3 * slab);
        zsolve_part_kernel<32, 2><<<grid, hs.L * hs.S, ds, st>>>(w, zp, hs.S, hs.L, h);
        if (p->singular && cudaStreamWaitEvent(st, p->ev_join, 0) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    } else if (p->bcz != PP_BC_PERIODIC) {
        // two-sweep Thomas; checkpoint table in shared memory: ceil(ceil(nz / 2) / CB) x TH doubles per CTA.
        // Lines beyond 4096 rows that the two-level partition does not take (nz not a multiple of 256) run with
        // 32 threads per CTA so that their 512 checkpoints per system still fit: slow, but every nz <= 16384 solves.
#define PP_ZT_LAUNCH(C, T)                                                                           \
        do {                                                                                         \
            const size_t ds = (size_t)(((p->nz + 1) / 2 + C - 1) / C) * T * sizeof(double) + PP_Z_DSMEM; \
            if (int rc = set_smem(zsolve_thomas_kernel<C, T>, ds)) return rc;                        \
            zsolve_thomas_kernel<C, T><<<(unsigned)((plane + T - 1) / T), T, ds, st>>>(w, zp);       \
        } while (0)
        if (p->nz > 64 * Z_MAX_CK) PP_ZT_LAUNCH(16, 32);
        else
#ifdef PP_Z_TH
        PP_ZT_LAUNCH(PP_Z_CB, PP_Z_TH);
#else
        PP_ZT_LAUNCH(PP_Z_CB, 128);
#endif
#undef PP_ZT_LAUNCH
    } else {
        // periodic z that the partitioned kernels do not take: Sherman-Morrison, three sweeps; two checkpoint
        // tables [ceil(nz / CB)][TH] in shared memory (at most 256 checkpoints x 32 threads, or 64 x 64)
#define PP_Z_LAUNCH(C, T)                                                                        \
        do {                                                                                     \
            const size_t ds = 2 * (size_t)((p->nz + C - 1) / C) * T * sizeof(double);            \
            if (int rc = set_smem(zsolve_cyclic_kernel<C, T>, ds)) return rc;                    \
            zsolve_cyclic_kernel<C, T><<<(unsigned)((plane + T - 1) / T), T, ds, st>>>(w, zp);   \
        } while (0)
        if (p->nz <= 16 * Z_MAX_CK)      PP_Z_LAUNCH(16, 64);
        else if (p->nz <= 32 * Z_MAX_CK) PP_Z_LAUNCH(32, 64);
        else if (p->nz <= 32 * 256)      PP_Z_LAUNCH(32, 32);
        else                             PP_Z_LAUNCH(64, 32);
#undef PP_Z_LAUNCH
    }
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}

}  // namespace pp

// ------------------------------------------------------------------------------------------------------------------
// pp_zsolve_static (include/pittpack_b200.h): the z solve (a7-a8) for callers that must not allocate device memory.
//
// Who that is: code running where a cudaMalloc is off limits -- a host application that handed all of the GPU's memory
// to its own pool at start-up and forbids the runtime allocator afterwards, a plug-in that is only ever given buffers,
// a latency-critical loop (cudaMalloc and cudaFree synchronise the whole device), or a process that is close to
// out of memory and cannot afford a plan.  Every other entry point of this library needs a pp_plan, and
// pp_plan_create uploads its tables with cudaMalloc.  This one takes no plan: the caller passes the grid, the two
// shift tables and the right-hand sides, and the only memory the kernel needs beyond those -- the work line of the
// singular (kx, ky) = (0, 0) system (zero_mode_line, pp_zsolve.cuh) -- is the fixed array below, which is part of the
// loaded library image: PP_STATIC_MAX_NZ doubles (32 KiB) on every GPU that loads the library, until the process exits.
//
// The kernel is the two-sweep Thomas kernel of the plan path (zsolve_thomas_kernel<16, 128>, the one PP_Z_SWEEP
// selects), unchanged; only where its scratch pointer comes from differs.  It lives in this file because the kernel
// templates of pp_zsolve.cuh can be included by one translation unit only.
namespace {

// The work line.  In HOST code this name is only a handle for the runtime (cudaGetSymbolAddress, cudaMemcpyToSymbol):
// its host-side address is not a device address and must never be handed to a kernel.  static_setup() below asks the
// runtime for the real address, once per device.
static __device__ __align__(256) double g_static_zero_line[PP_STATIC_MAX_NZ];

constexpr int CB = 16, TH = 128;                      // checkpoint spacing and threads per CTA, as pp_launch_z.cu
constexpr int MAX_DEVICES = 64;

constexpr size_t smem_bytes(int nz) { return (size_t)(((nz + 1) / 2 + CB - 1) / CB) * TH * sizeof(double); }

std::mutex g_static_mutex;
double *g_static_addr[MAX_DEVICES];                   // device address of g_static_zero_line per device; NULL: not set up yet

// Once per device, with that device current: the address of the work line on this device, and the kernel's opt-in
// to the dynamic shared memory of the longest line (a function attribute; no device memory is allocated).
int static_setup(int dev, double **line) {
    if (dev < 0 || dev >= MAX_DEVICES) return PP_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        double *ptr = nullptr;
        if (cudaGetSymbolAddress((void **)&ptr, g_static_zero_line) != cudaSuccess || !ptr) {
            cudaGetLastError();
            return PP_ERR_CUDA;
        }
        // through the library's registry of per-kernel limits, so that a plan using the same kernel never lowers it again
        if (int rc = pp::set_smem_once((const void *)pp::zsolve_thomas_kernel<CB, TH>, smem_bytes(PP_STATIC_MAX_NZ))) return rc;
        g_static_addr[dev] = ptr;
    }
    *line = g_static_addr[dev];
    return PP_SUCCESS;
}

}  // namespace

extern "C" int pp_zsolve_static(double *w, int nx, int ny, int nz, int bc_z, int zero_mode, double scale,
                                const double *sx, const double *sy, void *stream) {
    // argument checks first: none of them needs a device
    if (!w || !sx || !sy) return PP_ERR_NULL;
    if (nx < 1 || ny < 1 || nz < 2) return PP_ERR_INVALID_ARG;
    if (bc_z != PP_BC_NEUMANN && bc_z != PP_BC_DIRICHLET) return PP_ERR_INVALID_ARG;      // periodic z: not served here
    if (zero_mode != PP_ZERO_MODE_NONE && zero_mode != PP_ZERO_MODE_ZERO_MEAN && zero_mode != PP_ZERO_MODE_PIN_PLANE0)
        return PP_ERR_INVALID_ARG;
    if (zero_mode != PP_ZERO_MODE_NONE && bc_z != PP_BC_NEUMANN) return PP_ERR_INVALID_ARG; // a Dirichlet axis: never singular
    if (!std::isfinite(scale)) return PP_ERR_INVALID_ARG;
    if (nz > PP_STATIC_MAX_NZ) return PP_ERR_STATIC_LIMIT;                                  // the fixed work line is this long
    if (((uintptr_t)w & 7) || ((uintptr_t)sx & 7) || ((uintptr_t)sy & 7)) return PP_ERR_INVALID_ARG;
    const long long plane = (long long)nx * ny;
    if ((plane + TH - 1) / TH > (long long)INT_MAX) return PP_ERR_INVALID_ARG;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PP_ERR_CUDA; }
    double *line = nullptr;
    if (int rc = static_setup(dev, &line)) return rc;

    pp::ZParams zp;
    zp.nx = nx; zp.ny = ny; zp.nz = nz;
    zp.bcz = bc_z;
    zp.singular = zero_mode;
    zp.scale = scale;
    zp.sx = sx; zp.sy = sy;
    zp.zero_scratch = line;            // the device address from cudaGetSymbolAddress, not the symbol's host-side name
    zp.batch_stride = 0;
    pp::zsolve_thomas_kernel<CB, TH><<<(unsigned)((plane + TH - 1) / TH), TH, smem_bytes(nz), (cudaStream_t)stream>>>(w, zp);
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}
