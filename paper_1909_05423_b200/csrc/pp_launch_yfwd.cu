// y-pass launchers, forward (a4-a6): one instantiation per supported transform length, in place and
// (slab decomposition) with rows stored to their owner ranks' pencil blocks.
#include "pp_plan.h"
#include "pp_ypass.cuh"

namespace pp {

template <int N>
int launch_y_fwd(double *w, int nxh, int nz, int bc, int complex_cols, const double2 *tw, const double2 *ptw,
                 const YRows *rows, cudaStream_t st, YMapSlot *slot) {
    using Y = YCfg<N>;
    const dim3 grid((unsigned)((nxh + Y::T - 1) / Y::T), (unsigned)nz);
    if constexpr (YTma<N>::ON) {
        if (!rows && !YStaged<N>::ON) {
            // TMA-staged tiles: descriptors of this array (they hold its address: built on the host, kept in the plan
            // while the same array comes back)
            static_assert(sizeof(YTmaMaps) <= sizeof(slot->maps) && alignof(YTmaMaps) <= alignof(YMapSlot), "YMapSlot holds a YTmaMaps");
            YTmaMaps &maps = *reinterpret_cast<YTmaMaps *>(slot->maps);
            bool ok = slot->w == (const void *)w && slot->planes == nz && slot->bc == bc;
            if (!ok) {
                ok = tma_make_rows_map(&maps.all, (const double2 *)w, nxh, N, nz, 0, 1, N, Y::T, y_tma_box_rows(N));
                if (bc != BC_P)
                    ok = ok && tma_make_rows_map(&maps.even, (const double2 *)w, nxh, N, nz, 0, 2, N / 2, Y::T, y_tma_box_rows(N)) &&
                         tma_make_rows_map(&maps.odd, (const double2 *)w, nxh, N, nz, 1, 2, N / 2, Y::T, y_tma_box_rows(N));
                slot->w = ok ? (const void *)w : nullptr;
                slot->planes = nz;
                slot->bc = bc;
            }
            if (ok) {                       // (a driver without tensor maps: the plain kernel below)
                auto k = ypass_fwd_tma_kernel<N>;
                if (int rc = set_smem(k, Y::SMEM)) return rc;
                k<<<grid, Y::THREADS, Y::SMEM, st>>>((double2 *)w, nxh, bc, complex_cols, tw, ptw, maps);
                return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
            }
        }
    }
    if constexpr (YStaged<N>::ON) {      // (constexpr: the staged kernels exist only in a build that asks for them, -DPP_Y_STAGED_MIN=..)
      if (!rows) {
        // persistent staged kernel: one wave of resident CTAs walks over all tiles
        using S = YStaged<N>;
        auto k = ypass_staged_kernel<N, true>;
        if (int rc = set_smem(k, S::SMEM)) return rc;
        static int sms = 0;
        if (!sms) {
            int dev = 0;
            if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
                cudaGetLastError();
                sms = 0;
                return PP_ERR_CUDA;
            }
        }
        const long long total = (long long)grid.x * grid.y, resident = (long long)sms * S::PER_SM;
        k<<<(unsigned)(total < resident ? total : resident), Y::THREADS, S::SMEM, st>>>((double2 *)w, nxh, nz, bc, complex_cols, tw, ptw);
        return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
      }
    }
    if (rows) {
        auto k = ypass_fwd_slab_kernel<N>;
        if (int rc = set_smem(k, Y::SMEM)) return rc;
        k<<<grid, Y::THREADS, Y::SMEM, st>>>((double2 *)w, nxh, bc, complex_cols, tw, ptw, *rows);
    } else {
        auto k = ypass_fwd_kernel<N>;
        if (int rc = set_smem(k, Y::SMEM)) return rc;
        k<<<grid, Y::THREADS, Y::SMEM, st>>>((double2 *)w, nxh, bc, complex_cols, tw, ptw);
    }
    return cudaGetLastError() == cudaSuccess ? PP_SUCCESS : PP_ERR_CUDA;
}

int run_y_fwd(const pp_plan *p, double *w, const YRows *rows, cudaStream_t st, int z0, int nzs) {
    if (nzs < 0) nzs = p->nz;
    w += (size_t)z0 * p->nx * p->ny;
    const int complex_cols = (p->bcx == PP_BC_PERIODIC && p->bcy == PP_BC_PERIODIC) ? 1 : 0;
#define CALL_Y(NN) launch_y_fwd<NN>(w, p->nx / 2, nzs, p->bcy, complex_cols, p->tw_y, p->ptw_y, rows, st, &const_cast<pp_plan *>(p)->ymap[0])
    PP_DISPATCH_N(p->ny, CALL_Y)
#undef CALL_Y
}

}  // namespace pp
