/*
 * fsw_sweep_dispatch.cu -- picks the sweep-kernel instantiation (window size, view count) of a launch; the
 * instantiations themselves live in one object per (window, view count), fsw_sweep_inst.cu.
 */
#include "fsw_sweep.cuh"

#define FSW_DECL(w, n)                                                                                          \
    cudaError_t fsw_launch_sweep_w##w##_v##n(const FswSweepArgs& args, int variant, int grid, cudaStream_t stream); \
    cudaError_t fsw_prepare_sweep_w##w##_v##n();
#define FSW_DECL_SMALL(w) FSW_DECL(w, 0) FSW_DECL(w, 1) FSW_DECL(w, 2) FSW_DECL(w, 3) FSW_DECL(w, 4)
#define FSW_DECL_LARGE(w) FSW_DECL(w, 0) FSW_DECL(w, 1) FSW_DECL(w, 2)
FSW_DECL_SMALL(3) FSW_DECL_SMALL(5) FSW_DECL_SMALL(7) FSW_DECL_SMALL(9)
FSW_DECL_LARGE(11) FSW_DECL_LARGE(13) FSW_DECL_LARGE(15)

#define FSW_CASE(w, n) \
    case n: return prep ? fsw_prepare_sweep_w##w##_v##n() : fsw_launch_sweep_w##w##_v##n(args, variant, grid, stream);
#define FSW_WINDOW_SMALL(w)                                                                    \
    case w:                                                                                    \
        switch (fsw::nvt_for<w>(n_views, best_k)) { FSW_CASE(w, 0) FSW_CASE(w, 1) FSW_CASE(w, 2) FSW_CASE(w, 3) FSW_CASE(w, 4) } \
        break;
#define FSW_WINDOW_LARGE(w)                                                    \
    case w:                                                                    \
        switch (fsw::nvt_for<w>(n_views, best_k)) { FSW_CASE(w, 0) FSW_CASE(w, 1) FSW_CASE(w, 2) } \
        break;

static cudaError_t route(int window, int n_views, int best_k, bool prep, const FswSweepArgs& args, int variant, int grid, cudaStream_t stream) {
    switch (window) {
        FSW_WINDOW_SMALL(3) FSW_WINDOW_SMALL(5) FSW_WINDOW_SMALL(7) FSW_WINDOW_SMALL(9)
        FSW_WINDOW_LARGE(11) FSW_WINDOW_LARGE(13) FSW_WINDOW_LARGE(15)
        default: break;
    }
    return cudaErrorInvalidValue;
}

cudaError_t fsw_launch_sweep(int window, const FswSweepArgs& args, int variant, int grid, cudaStream_t stream) {
    return route(window, args.n_views, args.best_k, false, args, variant, grid, stream);
}

/* sets the shared-memory attribute of every variant that can serve calls with this window and view count */
cudaError_t fsw_prepare_sweep(int window, int n_views) {
    static const FswSweepArgs dummy = {};
    cudaError_t e = route(window, n_views, 0, true, dummy, 0, 0, nullptr);
    if (e == cudaSuccess && n_views > 1) e = route(window, n_views, 1, true, dummy, 0, 0, nullptr); /* the best-k variant */
    return e;
}

FswSweepGeometry fsw_sweep_geometry(int window, int n_views) {
    switch (window) {
        case 3: return fsw::geometry_win<3>(n_views);
        case 5: return fsw::geometry_win<5>(n_views);
        case 7: return fsw::geometry_win<7>(n_views);
        case 9: return fsw::geometry_win<9>(n_views);
        case 11: return fsw::geometry_win<11>(n_views);
        case 13: return fsw::geometry_win<13>(n_views);
        default: return fsw::geometry_win<15>(n_views);
    }
}
