/*
 * fsw_sweep_inst.cu -- one instantiation of the sweep kernel per matching-window size.
 * Compiled once per window with -DFSW_WIN=<w> (w odd, 3..15) so the instantiations build in parallel.
 */
#include "fsw_sweep.cuh"

#ifndef FSW_WIN
#error "compile with -DFSW_WIN=<odd window size>"
#endif

#define FSW_CAT2(a, b) a##b
#define FSW_CAT(a, b) FSW_CAT2(a, b)

cudaError_t FSW_CAT(fsw_launch_sweep_w, FSW_WIN)(const FswSweepArgs& args, int variant, int grid, cudaStream_t stream) {
    return fsw::launch_sweep_win<FSW_WIN>(args, variant, grid, stream);
}
cudaError_t FSW_CAT(fsw_prepare_sweep_w, FSW_WIN)() { return fsw::prepare_sweep_win<FSW_WIN>(); }
FswSweepGeometry FSW_CAT(fsw_geometry_sweep_w, FSW_WIN)(int n_views) { return fsw::geometry_win<FSW_WIN>(n_views); }
