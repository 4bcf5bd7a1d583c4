// Internal header of the library's translation units (not part of the C ABI): the plan structure and the
// per-pass launchers.  One .cu per pass family so that the instantiations compile in parallel:
//   pp_api.cu (plan, tables, C ABI) | pp_launch_x.cu | pp_launch_yfwd.cu | pp_launch_yinv.cu | pp_launch_z.cu |
//   pp_launch_fused.cu
#pragma once
#include "../../include/pittpack_b200.h"

#include <cuda_runtime.h>

#include "pp_fft.cuh"

namespace pp {
struct YRows;
}

// Tensor maps of the y passes (pp_tma.cuh) hold the address of the array they describe: they are encoded on the host, by
// the driver, and kept here per direction for as long as the same array, plane count and boundary condition come back --
// the usual case (a caller solving in the same buffers) then pays no cuTensorMapEncodeTiled on its launch path.
// `maps` is a YTmaMaps (pp_ypass.cuh; three CUtensorMap of 128 bytes, 64-byte aligned), opaque here.
struct alignas(64) YMapSlot {
    unsigned char maps[3 * 128];
    const void *w;             // array the maps describe (NULL: empty slot)
    int planes, bc;
};

struct pp_plan {
    YMapSlot ymap[2];          // [0] forward, [1] inverse y pass
    int nx, ny, nz;
    double dx, dy, dz;
    int bcx, bcy, bcz;
    int device;
    int num_sms;
    int singular;
    double scale;
    double2 *tw_x, *tw_y;      // per-stage FFT twiddle tables (pp_fft.cuh, tw_stage_offset)
    double2 *tw_xi;            // ... of the inverse x pass (== tw_x unless its radix schedule differs)
    double2 *ptw_x, *ptw_y;    // exp(-i pi m / (2n)), m in [0, n]
    double *sx, *sy;           // dz^2 lam / h^2 per packed position
    double *zero_scratch;      // [Z_MAX_BATCH][nz]
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
    int fused_per_sm[2];       // resident CTAs per SM of the fused forward / inverse kernel (0: not yet asked)
    double *hier_scratch;      // [4][nz / 256][nx ny]: interface values of the two-level z solve (long lines only)
    // x/y slab pipeline (pp_plan_set_xy_pipeline): the x and y passes run slab by slab on two streams, the y pass of
    // slab k beside the x pass of slab k+1, so that the intermediate slab is still in L2 when it is read back
    static constexpr int MAX_PIPE = 128;
    int xy_pipeline;           // planes per slab (0: off)
    cudaStream_t pipe;
    cudaEvent_t ev_pipe[MAX_PIPE], ev_pipe_join;
    cudaStream_t side;         // long singular lines only: the zero-mode line is solved beside the two-level passes
    cudaEvent_t ev_fork, ev_join;
    cudaEvent_t ev[PP_NUM_KERNELS + 1];
};

namespace pp {

// Opt a kernel in to more than 48 KB of dynamic shared memory -- once per (device, kernel) and size reached: pp_solve
// itself then only launches (no attribute call on the launch path of the small, latency-bound grids, and
// nothing but launches inside a stream capture after the first solve).  Defined in pp_api.cu.
int set_smem_once(const void *kernel, size_t smem);
template <class K>
inline int set_smem(K kernel, size_t smem) { return smem <= 48 * 1024 ? PP_SUCCESS : set_smem_once((const void *)kernel, smem); }

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


// the five passes (a1-a10 of SURVEY.md 8(a)); every launcher is stream-ordered and returns a PP_* status
// z0, nzs: the planes [z0, z0 + nzs) only (nzs < 0: all of them)
int run_x(const pp_plan *p, bool fwd, const double *in, double *out, cudaStream_t st, int z0 = 0, int nzs = -1);
int run_y_fwd(const pp_plan *p, double *w, const YRows *slab_rows, cudaStream_t st, int z0 = 0, int nzs = -1);   // slab_rows: see pp_ypass.cuh, or NULL
int run_y_inv(const pp_plan *p, double *w, const YRows *slab_rows, cudaStream_t st, int z0 = 0, int nzs = -1);
int run_z(const pp_plan *p, double *w, cudaStream_t st, int nbatch = 1);   // nbatch grids, nx ny nz doubles apart
int run_fused(const pp_plan *p, bool fwd, const double *in, double *u, cudaStream_t st);
bool fusion_supported(int nx, int ny);
bool zpart_range_ok(const pp_plan *p, int R);
bool zpart_single_level(const pp_plan *p);     // does a one-pass partitioned z kernel (one CTA or one cluster per line) take this plan
bool zpart_cluster(const pp_plan *p);          // ... the cluster kernel (by the plan's z_algorithm: where it pays, or wherever it applies)
bool zpart_cluster_possible(const pp_plan *p);

}  // namespace pp
