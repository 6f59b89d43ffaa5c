// shg_launch.h -- launcher prototypes shared by shg_inst.cu (one object per line length) and shg_api.cu.
#pragma once

#include <cuda_runtime.h>

namespace shg {

struct Params;

struct LaunchInfo {
    int rows_per_item;    // HG: rows (both fields) per row-pass item
    int cols_per_item;    // SC: columns per column-pass strip
    int warps;            // warps per CTA
    int row_slots;        // slots per CTA that can take row items (warps, or warp pairs at N = 1024)
    int col_teams;        // teams per CTA that can take strips
    int team_warps;       // warps per team
    int fft_r, fft_m;     // line length = fft_r * fft_m; twiddle table layout [fft_r][fft_m]
};

#define SHG_DECLARE_N(N)                                                                                   \
    cudaError_t launch_row_##N(const Params& P, int mode, int n, int hsel, bool prec, int grid,            \
                               cudaStream_t st);                                                            \
    cudaError_t launch_col_##N(const Params& P, int hsel, bool prec, int grid, cudaStream_t st);           \
    cudaError_t launch_persist_##N(const Params& P, bool prec, int grid, cudaStream_t st);                 \
    cudaError_t launch_cluster_##N(const Params& P, int csize, bool launch, int* max_clusters,             \
                                   cudaStream_t st);                                                        \
    LaunchInfo launch_info_##N();

// Records a failed CUDA call as the message behind shg_strerror(SHG_ECUDA) and returns SHG_ECUDA (shg_api.cu);
// lets the other translation units of the library (shg_static.cu) report through the same channel.
int record_cuda_error(cudaError_t e, const char* what);

SHG_DECLARE_N(64)
SHG_DECLARE_N(128)
SHG_DECLARE_N(256)
SHG_DECLARE_N(512)
SHG_DECLARE_N(1024)

}  // namespace shg
