// x-pass launchers (a1-a3, a10): one instantiation per supported transform length.
#include "pp_plan.h"
#include "pp_xpass.cuh"

namespace pp {

template <int N>
int launch_x(bool fwd, const double *in, double *out, long long npairs, int bc, const double2 *tw, const double2 *twi,
             const double2 *ptw, cudaStream_t st) {
    using XF = XCfg<N, false>;
    using XI = XCfg<N, true>;
    auto kf = xpass_fwd_kernel<N>;
    auto ki = xpass_inv_kernel<N>;
    if (fwd) {
        if (int rc = set_smem(kf, XF::SMEM)) return rc;
        kf<<<(unsigned)((npairs + XF::T - 1) / XF::T), XF::THREADS, XF::SMEM, st>>>(in, out, npairs, bc, tw, ptw);
    } else {
        if (int rc = set_smem(ki, XI::SMEM)) return rc;
        ki<<<(unsigned)((npairs + XI::T - 1) / XI::T), XI::THREADS, XI::SMEM, st>>>(in, out, npairs, bc, twi, ptw);
    }
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}

int run_x(const pp_plan *p, bool fwd, const double *in, double *out, cudaStream_t st, int z0, int nzs) {
    if (nzs < 0) nzs = p->nz;
    const size_t off = (size_t)z0 * p->nx * p->ny;
    in += off;
    out += off;
    const long long npairs = (long long)p->ny * nzs / 2;
#define CALL_X(NN) launch_x<NN>(fwd, in, out, npairs, p->bcx, p->tw_x, p->tw_xi, p->ptw_x, st)
    PP_DISPATCH_N(p->nx, CALL_X)
#undef CALL_X
}


}  // namespace pp
