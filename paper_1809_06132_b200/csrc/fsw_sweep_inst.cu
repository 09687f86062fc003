/*
 * fsw_sweep_inst.cu -- the instantiations of the sweep kernel for one matching-window size and one view count.
 * Compiled once per (window, view count) with -DFSW_WIN=<w> (odd, 3..15) -DFSW_NVT=<n> (1..4 views unrolled, 0 = the
 * run-time view loop) so that the objects build in parallel.
 */
#include "fsw_sweep.cuh"

#if !defined(FSW_WIN) || !defined(FSW_NVT)
#error "compile with -DFSW_WIN=<odd window size> -DFSW_NVT=<0..4>"
#endif

#define FSW_CAT4_(a, b, c, d) a##b##c##d
#define FSW_CAT4(a, b, c, d) FSW_CAT4_(a, b, c, d)

cudaError_t FSW_CAT4(fsw_launch_sweep_w, FSW_WIN, _v, FSW_NVT)(const FswSweepArgs& args, int variant, int grid, cudaStream_t stream) {
    return fsw::SweepInst<FSW_WIN, FSW_NVT>::launch(args, variant, grid, stream);
}
cudaError_t FSW_CAT4(fsw_prepare_sweep_w, FSW_WIN, _v, FSW_NVT)() { return fsw::SweepInst<FSW_WIN, FSW_NVT>::prepare(); }
