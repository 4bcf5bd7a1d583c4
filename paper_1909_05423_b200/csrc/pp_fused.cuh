// Plane-wise fusion of the x and y passes through the L2 cache.
//
// The x pass and the y pass of one z plane touch the same nx*ny doubles (2 MiB at 512 x 512), and
// the 2-D transform of a plane needs nothing from any other plane (the transforms
// act "in the x and y directions" of every xy plane independently).  Run as two kernels, the plane
// goes out to HBM after the x pass and comes back for the y pass.  Here both passes are tasks of one
// persistent kernel, ordered so that the y tasks of a plane are handed out shortly after its x
// tasks: the intermediate plane is written into L2 by the x tasks, read back from L2 by the y tasks
// and overwritten in L2 before it is ever evicted -- HBM sees one read and one write per point for
// the pair of passes (16 B/point instead of 32).  On one GPU this is what is left of the paper's
// chunk exchange between the x and y transforms.
//
// Scheduling.  Tasks are claimed by ticket (one atomicAdd per CTA and task) in the order
//     A(0) .. A(LAG-1) | A(LAG) B(0) | A(LAG+1) B(1) | ... | B(nz-LAG) .. B(nz-1)
// where A(z) are the NA first-phase tasks of plane z and B(z) its NB second-phase tasks
// (forward: A = x tiles, B = y tiles; inverse: A = y tiles, B = x tiles).  A B task waits until
// done[z] == NA; every A task it can wait for has a smaller ticket, i.e. is already running or
// finished on a resident CTA -- or is the prefetched next task of a CTA whose current task has a
// smaller ticket still -- so the unfinished task with the smallest ticket can always run and the
// wait cannot deadlock.  LAG is chosen so that the wait is
// normally over before it starts.  `sync` = [ticket, done[0..nz)], zeroed by the host before launch.
#pragma once
#include "pp_ypass.cuh"

namespace pp {

#ifndef PP_FUSE_LDCG
#define PP_FUSE_LDCG true   // second-phase tiles read with ld.global.cg (L2): their input comes from other SMs
#endif

struct FusedParams {
    int nz, nxh;            // planes, double2 per row
    int na, nb;             // first-/second-phase tasks per plane
    int lag;                // planes the second phase trails the first by (1 <= lag <= nz)
    int bcx, bcy, complex_cols;
    long long pairs_per_plane;
    int *sync;              // [1 + nz]
};

struct FusedTask {
    int phase, z, idx;
};

__device__ __forceinline__ FusedTask fused_decode(int t, const FusedParams &p) {
    const int head = p.lag * p.na;
    if (t < head) return {0, t / p.na, t % p.na};
    t -= head;
    const int per = p.na + p.nb, mid = (p.nz - p.lag) * per;
    if (t < mid) {
        const int s = t / per, r = t % per;
        if (r < p.na) return {0, p.lag + s, r};
        return {1, s, r - p.na};
    }
    t -= mid;
    return {1, p.nz - p.lag + t / p.nb, t % p.nb};
}

__device__ __forceinline__ int ld_acquire_gpu(const int *p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// The four tile bodies as real (not inlined) functions: each gets its own register allocation, and
// nothing of the scheduler's state is live inside them.
template <int N, int TX>
__device__ __noinline__ void fused_xfwd(const double *in, double *u, long long pair0, long long pend, int bc,
                                        const double2 *tw, const double2 *ptw, double2 *smem) {
    xfwd_tile<N, TX>(in, u, pair0, pend, bc, tw, ptw, smem);
}
template <int N, int TX>
__device__ __noinline__ void fused_xinv(double *u, long long pair0, long long pend, int bc,
                                        const double2 *tw, const double2 *ptw, double2 *smem) {
    xinv_tile<N, TX, PP_FUSE_LDCG>(u, u, pair0, pend, bc, tw, ptw, smem);
}
template <int N>
__device__ __noinline__ void fused_yfwd(double2 *u, int nxh, int bc, int cc, const double2 *tw, const double2 *ptw,
                                        int bx, int z, double2 *smem) {
    yfwd_tile<N, PP_FUSE_LDCG>(u, nxh, bc, cc, tw, ptw, bx, z, smem);
}
template <int N>
__device__ __noinline__ void fused_yinv(double2 *u, int nxh, int bc, int cc, const double2 *tw, const double2 *ptw,
                                        int bx, int z, double2 *smem) {
    yinv_tile<N>(u, nxh, bc, cc, tw, ptw, bx, z, smem);
}

// FWD_DIR: x forward tiles then y forward tiles (in -> u, then in place);
// otherwise y inverse tiles then x inverse tiles (in place in u).
template <int N, bool FWD_DIR>
__global__ void __launch_bounds__(YCfg<N>::THREADS, YCfg<N>::MINB)
xy_fused_kernel(const double *in, double *u, FusedParams p,
                const double2 *__restrict__ tw_x, const double2 *__restrict__ ptw_x,
                const double2 *__restrict__ tw_y, const double2 *__restrict__ ptw_y) {
    using Y = YCfg<N>;
    constexpr int TX = Y::THREADS / Y::P;               // row pairs per x tile (= Y::T)
    extern __shared__ double2 smem[];
    __shared__ int s_ticket;
    int *ticket = p.sync, *done = p.sync + 1;
    const int total = p.nz * (p.na + p.nb);
    if (threadIdx.x == 0) s_ticket = atomicAdd(ticket, 1);
    __syncthreads();
    int t = s_ticket;
    while (t < total) {
        // claim the next task now: the atomic's round trip hides behind this tile
        int next = 0;
        if (threadIdx.x == 0) next = atomicAdd(ticket, 1);
        const FusedTask k = fused_decode(t, p);
        if (k.phase == 1) {
            if (threadIdx.x == 0) {
                while (ld_acquire_gpu(done + k.z) < p.na) __nanosleep(100);
            }
            __syncthreads();
        }
        const bool xtile = FWD_DIR ? (k.phase == 0) : (k.phase == 1);
        if (xtile) {
            const long long pair0 = (long long)k.z * p.pairs_per_plane + (long long)k.idx * TX;
            const long long pend = (long long)(k.z + 1) * p.pairs_per_plane;     // tiles do not straddle planes
            if (FWD_DIR) fused_xfwd<N, TX>(in, u, pair0, pend, p.bcx, tw_x, ptw_x, smem);
            else         fused_xinv<N, TX>(u, pair0, pend, p.bcx, tw_x, ptw_x, smem);
        } else {
            if (FWD_DIR) fused_yfwd<N>((double2 *)u, p.nxh, p.bcy, p.complex_cols, tw_y, ptw_y, k.idx, k.z, smem);
            else         fused_yinv<N>((double2 *)u, p.nxh, p.bcy, p.complex_cols, tw_y, ptw_y, k.idx, k.z, smem);
        }
        __syncthreads();                                // the tile is done with smem; its stores are issued
        if (threadIdx.x == 0) {
            if (k.phase == 0) {
                __threadfence();
                atomicAdd(done + k.z, 1);
            }
            s_ticket = next;
        }
        __syncthreads();
        t = s_ticket;
    }
}

}  // namespace pp
