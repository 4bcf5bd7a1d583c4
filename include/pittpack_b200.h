/*
 * pittpack_b200 -- C ABI of the B200-native direct Poisson solver.
 *
 * What it computes (arxiv 1909.05423 "PittPack"; citations are lines of the paper text
 * PAPER.md): the solution u of the second-order 7-point finite-difference Poisson equation
 *
 *   (u[i+1,j,k]-2u[i,j,k]+u[i-1,j,k])/dx^2 + (..j..)/dy^2 + (..k..)/dz^2 = f[i,j,k]      (eq. 3)
 *
 * on a directionally-uniform cell-centred nx x ny x nz grid, with one
 * homogeneous boundary condition per axis imposed at the cell faces: periodic, Neumann
 * (zero normal derivative) or Dirichlet (zero value, ghost cell by linear
 * extrapolation).  Method: forward
 * FFT / DCT-II / DST-II along x and then y chosen by each axis' boundary condition
 * (Table 1), each built on a complex FFT with fused pre/post passes
 * (PAPER.md:103-107); one tridiagonal Thomas solve in z per (kx,ky) with the modified-
 * wavenumber diagonal of Table 2 -- Sherman-Morrison when z is periodic
 * -- and the zero-mode fix; then the inverse transforms.
 *
 * Everything on the path is a hand-written CUDA kernel for sm_100a, fp64 throughout.  There
 * is no cuFFT / cuSPARSE call and no CPU fallback: on a machine without a CUDA device every
 * entry point that needs one returns PP_ERR_CUDA.
 *
 * Memory convention: x fastest, idx = i + nx*(j + ny*k); as a tensor, shape (nz, ny, nx),
 * contiguous, float64.  The value at idx belongs to the cell centre ((i+1/2)dx, (j+1/2)dy,
 * (k+1/2)dz).
 *
 * Singular case (all three axes periodic or Neumann): f is projected to
 * zero mean and the zero-mean solution is returned (= the pseudo-inverse applied to f).
 *
 * Non-homogeneous Dirichlet face values g are the caller's job, folded into the source as
 * PAPER.md:163 describes:  f[boundary cell] -= 2 g / h^2.
 *
 * Threading: a plan may be reused indefinitely, from any host thread, but concurrent
 * pp_solve calls on ONE plan are not allowed (its tables are shared, its scratch is single).
 * All functions return a status code; none throws, none aborts.
 */
#ifndef PITTPACK_B200_H
#define PITTPACK_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pp_plan pp_plan; /* opaque; owns device tables and scratch */

/* One boundary condition per axis, applied on both faces (Table 2 has matched pairs only). */
enum { PP_BC_PERIODIC = 0, PP_BC_NEUMANN = 1, PP_BC_DIRICHLET = 2 };

enum {
    PP_SUCCESS = 0,
    PP_ERR_INVALID_ARG = 1,      /* non-positive size/spacing, unknown BC, misaligned or partially overlapping pointers */
    PP_ERR_UNSUPPORTED_SIZE = 2, /* nx or ny not a supported transform length, nz out of range (see pp_plan_create) */
    PP_ERR_ALLOC = 3,            /* host or device allocation failed */
    PP_ERR_CUDA = 4,             /* a CUDA runtime call or kernel launch failed (no device, bad stream, ...) */
    PP_ERR_NULL = 5,             /* a required pointer argument is NULL */
    PP_ERR_STATIC_LIMIT = 6      /* pp_zsolve_static: nz beyond PP_STATIC_MAX_NZ, the length of its built-in work line */
};

/* The five passes of one pp_solve and their order: the timing slots of pp_plan_last_kernel_ms.  By default each
 * is one kernel; a slot can hold several (two-level z solve) or none (x+y fusion): pp_plan_launches_per_solve. */
enum { PP_K_XFWD = 0, PP_K_YFWD = 1, PP_K_ZSOLVE = 2, PP_K_YINV = 3, PP_K_XINV = 4, PP_NUM_KERNELS = 5 };

/*
 * Create a plan for an nx x ny x nz grid with spacings dx, dy, dz and boundary conditions
 * bc_x, bc_y, bc_z (PP_BC_*).  Mirrors the paper's construction "PoissonGPU(n0,n1,n2)" +
 * "assignBoundary(bc)" (Listing 3).
 *   out      : host pointer receiving the handle (set to NULL on failure).
 *   nx, ny   : 2^k in [4, 2048], 3 * 2^k in [48, 1536] or 5 * 2^k in [80, 1280] (the hand-written FFT
 *              core; the 48-multiples are the paper's weak-scaling grids);  nz in [2, 16384], any
 *              boundary condition (16384: the paper's 64 x 64 x 16384 pencils).  Which z kernel
 *              serves which nz: pp_plan_set_z_algorithm.
 * Synchronous.  Builds the twiddle, post-twiddle and modified-wavenumber tables on the host
 * in extended precision and uploads them to the CURRENT device; the plan is bound to it.
 */
int pp_plan_create(pp_plan **out, int nx, int ny, int nz, double dx, double dy, double dz,
                   int bc_x, int bc_y, int bc_z);

/*
 * Solve A u = f  (the paper's "pittPack(P)").
 *   f, u   : DEVICE pointers to nx*ny*nz doubles, x fastest, 16-byte aligned, owned by the
 *            caller.  u == f (exact aliasing, in place) is allowed; any other overlap is
 *            PP_ERR_INVALID_ARG.  f is not modified unless u == f.
 *   stream : a cudaStream_t passed as void* (NULL = the legacy default stream).
 * Asynchronous and stream-ordered: enqueues its kernels (pp_plan_launches_per_solve) on `stream` -- one
 * small kernel of the long-line singular case runs on a plan-owned side stream, forked from and joined
 * back into `stream` by events, so the ordering seen by the caller is the same -- never
 * allocates, never synchronises.  Launch errors are returned; execution errors surface at
 * the caller's next synchronisation.  All passes run in place in u: no N-sized workspace.
 */
int pp_solve(const pp_plan *plan, const double *f, double *u, void *stream);

/*
 * Same solve with HOST buffers (nx*ny*nz doubles each; pinned memory recommended): copies
 * f to a plan-owned device buffer, solves in place, copies the result to u_host, all on
 * `stream`, then synchronises the stream before returning.  The device buffer is allocated
 * on first use (PP_ERR_ALLOC if that fails) and lives until pp_plan_destroy.
 */
int pp_solve_host(pp_plan *plan, const double *f_host, double *u_host, void *stream);

/*
 * nbatch independent solves with HOST buffers: right-hand side i is the i-th block of nx*ny*nz doubles of
 * f_host, its solution the i-th block of u_host (pinned memory recommended; the two may be the same buffer).
 * The copy-in of right-hand side i+1 and the copy-out of solution i-1 run beside the solve of i (two
 * plan-owned copy streams, a ring of three plan-owned device buffers, allocated on first use), so a long
 * batch costs one PCIe direction per solve instead of two.  Synchronises before returning.
 */
int pp_solve_host_batch(pp_plan *plan, const double *f_host, double *u_host, int nbatch, void *stream);

/*
 * nbatch independent solves with DEVICE buffers: right-hand side i is the i-th block of nx*ny*nz doubles of f, its
 * solution the i-th block of u (same rules as pp_solve: 16-byte aligned, u == f allowed, no partial overlap).  The
 * transforms of all right-hand sides run as ONE launch per pass (the x and y transforms act on every xy plane
 * independently: a batch is a taller stack of planes).  The z solves: where the one-CTA partitioned
 * kernel serves the plan (nz = 32m / 64m <= 512, 1024, 2048; not under PP_Z_SWEEP) up to 64 grids per launch, i.e.
 * 4 + ceil(nbatch / 64) launches in all; otherwise one z solve after the other, 4 + k nbatch launches with k the
 * z-solve launches of one pp_solve (pp_plan_launches_per_solve - 4) -- instead of (4 + k) nbatch.  A stack taller
 * than 65535 planes (the y passes put one plane per blockIdx.y) is cut into groups of floor(65535 / nz) grids, each
 * group launched as above; any nbatch with nz * nbatch < 2^31 is accepted.  The use the paper itself names is a
 * complex source, "two solves" for its real and imaginary part (reading R17), and small grids stop
 * being launch-bound.
 * Stream-ordered, no allocation, no synchronisation.  The x+y fusion / pipeline settings of the plan are ignored.
 */
int pp_solve_batch(const pp_plan *plan, const double *f, double *u, int nbatch, void *stream);

/* Free the plan and everything it owns.  NULL is a no-op returning PP_SUCCESS. */
int pp_plan_destroy(pp_plan *plan);

/* Device bytes the plan currently owns (tables + scratch + the host-solve staging buffer if created). */
size_t pp_plan_workspace_bytes(const pp_plan *plan);

/*
 * Per-pass timing for roofline reports.  With profiling enabled, pp_solve brackets each of
 * its PP_NUM_KERNELS passes with CUDA events on the caller's stream (no synchronisation).
 * pp_plan_last_kernel_ms synchronises on the last event and writes PP_NUM_KERNELS
 * durations in milliseconds (order PP_K_*) into ms_out (host pointer).
 */
int pp_plan_set_profiling(pp_plan *plan, int enable);
int pp_plan_last_kernel_ms(pp_plan *plan, float *ms_out);

/*
 * Which kernel solves the tridiagonal systems in z (PAPER.md:208-218 leaves the choice of
 * tridiagonal algorithm open and offers several).  Both compute the same
 * Thomas elimination of Algorithm 2 up to rounding order.
 *   PP_Z_AUTO      : partitioned where it applies, two-sweep otherwise (the default).
 *   PP_Z_SWEEP     : two-sweep Thomas, one thread per system, any nz; periodic z by
 *                    Sherman-Morrison.  (Beyond 4096 rows it runs 32 threads per CTA: a
 *                    fallback for line lengths the partition does not take, not a fast path.)
 *   PP_Z_PARTITION : each system cut into segments of 32 or 64 rows held in registers and
 *                    coupled through their interface unknowns (the reduction idea of CR-P,
 *                    PAPER.md:250-258, across the threads of one CTA); with periodic z the
 *                    interface chain closes on itself (a 2x2 closure instead of Sherman-Morrison's
 *                    second solve).  Needs nz = 32 m or 64 m (m <= 8), 1024 or 2048 -- or
 *                    nz = 256 m (2 <= m <= 64), where the same partition is applied on two levels
 *                    (super-segments of 256 rows, three kernels; with periodic z the chain of
 *                    super-segments closes on itself the same way); otherwise
 *                    PP_ERR_UNSUPPORTED_SIZE and the plan is left unchanged.  The partitioned kernels tabulate segment
 *                    determinants of magnitude up to (3 + max|s|)^R (R = 32 or 64 rows per
 *                    segment, s the spectral shift dz^2 (lam_x/dx^2 + lam_y/dy^2)); grids so
 *                    anisotropic that this could leave the fp64 range (dz/dx beyond ~90 with
 *                    R = 64, ~17000 with R = 32) are solved by the two-sweep kernel instead.
 *   PP_Z_CLUSTER   : nz = 256 m, 2 <= m <= 8, Neumann / Dirichlet z: the two levels of PP_Z_PARTITION in ONE
 *                    kernel -- the m CTAs of a line form a thread-block cluster, keep their super-segment in
 *                    registers and exchange its first and last unknown through distributed shared memory
 *                    (8 B read + 8 B written per point instead of 24).  PP_Z_AUTO picks it where it measured
 *                    faster (nz = 768, 1280 ... 2048 except 1024, at least 32768 lines); this value forces it
 *                    wherever it applies; otherwise PP_ERR_UNSUPPORTED_SIZE.
 */
enum { PP_Z_AUTO = 0, PP_Z_SWEEP = 1, PP_Z_PARTITION = 2, PP_Z_CLUSTER = 3 };
int pp_plan_set_z_algorithm(pp_plan *plan, int algorithm);

/*
 * Plane-wise fusion of the x and y passes.  The 2-D transform of one xy plane is independent of
 * every other plane.  With fusion enabled the x tiles and y tiles of a plane are
 * tasks of ONE persistent kernel, ordered so that a plane's intermediate spectrum stays in the L2
 * cache between its x and y pass: pp_solve then launches 3 kernels (x+y forward, z solve, y+x
 * inverse) and HBM sees 48 instead of 80 bytes per point.  Results are bit-identical to the
 * unfused path.  Needs nx == ny in {128, 256, 512}; otherwise PP_ERR_UNSUPPORTED_SIZE and the
 * plan is left unchanged.  With fusion on, pp_plan_last_kernel_ms reports the fused kernels' times
 * in the PP_K_XFWD and PP_K_XINV slots and 0 for PP_K_YFWD / PP_K_YINV.
 */
int pp_plan_set_xy_fusion(pp_plan *plan, int enable);

/*
 * The same idea with plain launches: the x and y passes run slab by slab (planes_per_slab z planes at a time), the
 * first pass of slab k on the caller's stream, the second on a plan-owned stream as soon as the first is done --
 * beside the first pass of slab k+1 -- so that a slab (planes_per_slab nx ny doubles; 32 MiB for 16 planes of
 * 512 x 512) is still in L2 when it is read back.  The caller's stream joins at the end: pp_solve stays
 * stream-ordered (and capturable).  Any grid; 0 switches it off (the default); more than 128 slabs ->
 * PP_ERR_INVALID_ARG.  Results are bit-identical.  Measured at 512 x 512 x 256: HBM traffic of a pair halves, its
 * time does not improve (0.36 against 0.33 ms for the two passes run one after the other): the passes are bound
 * by the SMs' shared-memory pipe, not by HBM.  Timing slots as with pp_plan_set_xy_fusion.
 */
int pp_plan_set_xy_pipeline(pp_plan *plan, int planes_per_slab);

/*
 * Non-homogeneous Dirichlet face values, moved to the right-hand side as PAPER.md:163 prescribes for
 * a ghost cell extrapolated linearly through the face value:  f[boundary cell] -= 2 g / h^2.
 * Call it on f before pp_solve (which solves the homogeneous problem); cells on an edge or a corner
 * receive every face's term.
 *   f                    : DEVICE pointer, nx*ny*nz doubles, modified in place.
 *   gx_lo, gx_hi         : DEVICE arrays [nz][ny] of values on the faces x = 0 / x = nx dx, or NULL.
 *   gy_lo, gy_hi         : [nz][nx] on y = 0 / y = ny dy, or NULL.   gz_lo, gz_hi : [ny][nx], or NULL.
 * A non-NULL face of an axis that is not Dirichlet is PP_ERR_INVALID_ARG.  Stream-ordered, no sync.
 */
int pp_fold_dirichlet(const pp_plan *plan, double *f, const double *gx_lo, const double *gx_hi,
                      const double *gy_lo, const double *gy_hi, const double *gz_lo, const double *gz_hi,
                      void *stream);

/*
 * Which solution of a singular problem (all three axes periodic or Neumann) is returned.  f is
 * projected to zero mean either way (second alternative); the solution is then fixed
 * up to a constant:
 *   PP_NULL_ZERO_MEAN  : zero volume mean, u = pinv(A) f (the default; what the oracle returns).
 *   PP_NULL_PIN_PLANE0 : the mean of the z = 0 plane is zero -- the paper's default ("keeping the
 *                        corner value which is the mean of the function at z=0 plane fixed",
 *                        PAPER.md:533).  Differs from the first by the constant mean_xy u(:,:,0).
 * No effect on non-singular plans.
 */
enum { PP_NULL_ZERO_MEAN = 0, PP_NULL_PIN_PLANE0 = 1 };
int pp_plan_set_null_space(pp_plan *plan, int convention);

/*
 * 1 if pp_plan_create accepts this grid (see its size rules), else 0.  Host-only: needs no device.
 * (Spacing-dependent refusals -- lines longer than 4096 on extremely anisotropic grids -- are not
 * covered: they need dx, dy, dz.)
 */
int pp_size_supported(int nx, int ny, int nz, int bc_z);

/*
 * Number of kernels one pp_solve launches with the plan's current settings: 5 by default (PP_K_*),
 * 3 with x+y fusion, +2 (+1 more when the problem is singular) when the z solve is the two-level
 * partition for long lines.  0 for a NULL plan.
 */
int pp_plan_launches_per_solve(const pp_plan *plan);

/*
 * ---- Slab decomposition over `world` GPUs (one process per GPU) -------------------------------
 *
 * The paper's pencil decomposition and all-to-all on NVLink, re-thought: rank r owns the z-slab of
 * nz/world planes [r nz/world, (r+1) nz/world) of f and u -- the x and y transforms are local to a slab --
 * and, for the z solve, the (kx, ky)-pencil of ny/world wavenumber rows ky in [q ny/world, (q+1) ny/world), all kx, all
 * nz planes (the tridiagonal systems are independent per (kx, ky)).  Pencil layout: [nz][ny/world][nx],
 * x fastest.  The two re-orientations are FUSED INTO THE y PASSES: the forward y pass stores each spectral row straight
 * into the pencil block of the rank that owns it, the inverse y pass loads its rows from there -- no pack / unpack
 * kernel, no staging.  The library never communicates by itself; it is given the addresses:
 *
 *   chunk(r -> q) = the nz/world planes of slab r restricted to the rows of pencil q: [nz/world][ny/world][nx] doubles,
 *   which is a contiguous piece of pencil q (planes r nz/world ...), starting at pencil_q + r * chunk_elems.
 *
 *   fwd_dst[q] : where THIS rank's forward pass writes chunk(rank -> q):  peer memory (pencil_q + rank * chunk_elems,
 *                mapped through CUDA IPC / a peer-enabled pointer), or chunk q of a local send buffer that an
 *                all-to-all (NCCL) then delivers -- the receive buffer of that all-to-all IS the pencil.
 *   inv_src[q] : where THIS rank's inverse pass reads chunk(rank <- q) of the solved pencils: peer memory again
 *                (pencil_q + rank * chunk_elems), or chunk q of the receive buffer of the return all-to-all, whose send
 *                buffer is the pencil itself.
 * Bytes crossing NVLink per GPU, per direction and per exchange: 8 N (world-1) / world^2.
 *
 * Call order per solve, with a cross-rank barrier on the stream where marked (the caller's job: an NCCL all-reduce,
 * or the all-to-all itself):
 *      pp_slab_forward(f_slab)  |barrier / all-to-all|  pp_slab_zsolve(pencil)  |barrier / all-to-all|  pp_slab_inverse(u_slab)
 *
 * Needs nz % world == 0, ny % world == 0, nz/world >= 2, world <= 16; sizes otherwise as pp_plan_create.
 * Singular problems: the (0,0) line lives on rank 0's pencil, which applies the zero-mode fix -- same result as one GPU.
 */
typedef struct pp_slab_plan pp_slab_plan;
int pp_slab_plan_create(pp_slab_plan **out, int world, int rank, int nx, int ny, int nz, double dx, double dy, double dz,
                        int bc_x, int bc_y, int bc_z);
int pp_slab_plan_destroy(pp_slab_plan *plan);
/* doubles in this rank's slab, = doubles in its pencil: nx ny nz / world;  and in one chunk: nx ny nz / world^2 */
size_t pp_slab_local_elems(const pp_slab_plan *plan);
size_t pp_slab_chunk_elems(const pp_slab_plan *plan);
/* fwd_dst, inv_src: HOST arrays of `world` DEVICE addresses (see above), copied into the plan.  May be called again. */
int pp_slab_set_exchange(pp_slab_plan *plan, double *const *fwd_dst, const double *const *inv_src);
/* x forward + y forward on the slab.  f_slab: nz/world planes (read only); work_slab: same size, holds the x spectrum
 * (f_slab == work_slab allowed).  The y pass writes through fwd_dst.  Stream-ordered, no sync. */
int pp_slab_forward(const pp_slab_plan *plan, const double *f_slab, double *work_slab, void *stream);
/* every tridiagonal system of this rank's pencil [nz][ny/world][nx], in place. */
int pp_slab_zsolve(const pp_slab_plan *plan, double *pencil, void *stream);
/* y inverse (reading through inv_src) + x inverse, result in u_slab (nz/world planes). */
int pp_slab_inverse(const pp_slab_plan *plan, double *u_slab, void *stream);

/*
 * ---- The z solve without a plan and without any allocation -----------------------------------------------------
 *
 * For callers that cannot allocate device memory: an application that gave the whole GPU to its own memory pool at
 * start-up and allows no cudaMalloc afterwards, a plug-in that only ever receives buffers, a time-critical loop (the
 * runtime allocator synchronises the device), a process too close to out-of-memory to afford a plan.  Everything else
 * in this header goes through a pp_plan, and pp_plan_create allocates.  pp_zsolve_static solves the tridiagonal
 * systems of step a7-a8 (Algorithm 1; diagonal of Table 2) with what the caller
 * passes in and one fixed work line of PP_STATIC_MAX_NZ doubles that is compiled into the library (32 KiB of every
 * GPU that loads the library, held until the process exits).  It calls no cudaMalloc / cudaFree and no routine that
 * allocates.  Same kernel and same arithmetic as a plan under PP_Z_SWEEP.
 *
 *   w         : DEVICE, nx*ny*nz doubles, x fastest: the right-hand sides after the forward x and y transforms;
 *               overwritten by the solutions.  System (ix, j) is the strided line w[ix + nx*(j + ny*k)], k = 0..nz-1.
 *   bc_z      : PP_BC_NEUMANN or PP_BC_DIRICHLET (first / last diagonal -1 + s / -3 + s).  Periodic z is not offered
 *               here: PP_ERR_INVALID_ARG.
 *   zero_mode : PP_ZERO_MODE_NONE, or -- when both transformed axes are periodic / Neumann and bc_z is Neumann, so
 *               that system (0, 0) is singular -- which solution of it to return: zero volume mean
 *               (what pp_solve returns by default) or zero value in plane 0 (PP_NULL_PIN_PLANE0).  Anything but
 *               NONE with a Dirichlet bc_z is PP_ERR_INVALID_ARG.
 *   scale     : every right-hand side is multiplied by this first (a plan uses dz^2 / (nx ny): Table 2's dz^2 and the
 *               normalisation of the inverse transforms).
 *   sx, sy    : DEVICE tables of nx and ny doubles, read only: the diagonal of system (ix, j) is -2 + sx[ix] + sy[j],
 *               i.e. sx[ix] = dz^2 lambda_x(k(ix)) / dx^2 with lambda from Table 2 and k(ix) the wavenumber stored at
 *               position ix (for this library's periodic x layout: k = 0, nx/2, 1, 1, 2, 2, ...), sy likewise.
 *               All entries <= 0, and < 0 for every system except a singular (0, 0).
 *   stream    : cudaStream_t as void*.  Asynchronous, stream-ordered, one kernel launch.
 *
 * Limit: nz <= PP_STATIC_MAX_NZ, else PP_ERR_STATIC_LIMIT and nothing is launched (longer lines need a plan).
 * First call on a device: it looks up the device address of the work line (cudaGetSymbolAddress) and raises the
 * kernel's shared-memory limit, once, with that device current.  Make that first call outside any stream capture.
 * The work line is shared by every call in the process and keeps whatever the last call left in it.  Nothing in it
 * has to start at zero -- the kernel writes each element before it reads it -- so calls that follow one another on a
 * stream need no clearing; but two calls with zero_mode != NONE that overlap on the GPU (different streams, other
 * threads, no ordering between them) write the same line and corrupt each other's (0, 0) system.  Order them.
 */
#define PP_STATIC_MAX_NZ 4096
enum { PP_ZERO_MODE_NONE = 0, PP_ZERO_MODE_ZERO_MEAN = 1, PP_ZERO_MODE_PIN_PLANE0 = 2 };
int pp_zsolve_static(double *w, int nx, int ny, int nz, int bc_z, int zero_mode, double scale,
                     const double *sx, const double *sy, void *stream);

/* Static, NUL-terminated description of a status code. */
const char *pp_strerror(int status);

/* Library version string, e.g. "pittpack_b200 0.1 (sm_100a)". */
const char *pp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PITTPACK_B200_H */
