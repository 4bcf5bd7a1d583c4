// Launcher of the opt-in plane-wise x+y fusion (pp_fused.cuh).
#include "pp_plan.h"
#include "pp_fused.cuh"

namespace pp {

// nx == ny in {128, 256, 512}: the sizes the fused x+y kernel is instantiated for (its x and y tiles share
// one CTA shape, i.e. one radix schedule)
bool fusion_supported(int nx, int ny) { return nx == ny && nx >= 128 && nx <= 512 && (nx & (nx - 1)) == 0; }

#ifndef PP_FUSE_LAG
#define PP_FUSE_LAG 0          // 0: derived from the number of resident CTAs
#endif

template <int N, bool FWD_DIR>
int launch_fused(const pp_plan *p, const double *in, double *u, cudaStream_t st) {
    using Y = YCfg<N>;
    static_assert(XCfg<N>::E == Y::E, "fused x+y tiles share one radix schedule");
    constexpr int TX = Y::THREADS / Y::P;
    auto kernel = xy_fused_kernel<N, FWD_DIR>;
    if (int rc = set_smem(kernel, Y::SMEM)) return rc;
    int &per_sm = const_cast<pp_plan *>(p)->fused_per_sm[FWD_DIR ? 0 : 1];      // resolved by the first fused solve
    if (per_sm < 1 &&
        (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, Y::THREADS, Y::SMEM) != cudaSuccess || per_sm < 1)) {
        per_sm = 0;
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
        default:   return PP_ERR_UNSUPPORTED_SIZE;
    }
}

}  // namespace pp
