// shg_inst.cu -- kernel instantiations and launchers for one line length SHG_N (compiled once per N so the
// sizes build in parallel).  Host code in shg_api.cu picks the launcher by nx / ny.
#ifndef SHG_N
#error "compile with -DSHG_N=<64|128|256|512|1024>"
#endif

#include "shg_device.cuh"
#if SHG_N <= 128
#include "shg_cluster.cuh"
#endif
#include "shg_launch.h"

namespace shg {

namespace {
constexpr int N = SHG_N;
using GE = Geo<N>;

template <typename K>
cudaError_t set_smem(K kernel, int bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

template <int MODE, bool PREC, bool HEAT = false>
cudaError_t launch_row_t(const Params& P, int n, int hsel, int grid, cudaStream_t st) {
    cudaError_t e = set_smem(k_row<N, MODE, PREC, HEAT>, GE::CTA_SMEM);
    if (e != cudaSuccess) return e;
    k_row<N, MODE, PREC, HEAT><<<grid, GE::THREADS, GE::CTA_SMEM, st>>>(P, n, hsel);
    return cudaGetLastError();
}

template <int MODE>
cudaError_t launch_row_paper_t(const Params& P, int n, int grid, cudaStream_t st) {
    cudaError_t e = set_smem(k_row_paper<N, MODE, true>, GE::CTA_SMEM);
    if (e != cudaSuccess) return e;
    k_row_paper<N, MODE, true><<<grid, GE::THREADS, GE::CTA_SMEM, st>>>(P, n);
    return cudaGetLastError();
}

template <bool PREC>
cudaError_t launch_col_t(const Params& P, int hsel, int grid, cudaStream_t st) {
    cudaError_t e = set_smem(k_col<N, PREC>, GE::CTA_SMEM);
    if (e != cudaSuccess) return e;
    k_col<N, PREC><<<grid, GE::THREADS, GE::CTA_SMEM, st>>>(P, hsel);
    return cudaGetLastError();
}

template <bool PREC, bool HEAT, bool TS = false>
cudaError_t launch_persist_t(const Params& P, int grid, cudaStream_t st) {
    const int smem = TS ? GE::CTA_SMEM_TAB : GE::CTA_SMEM + ((!HEAT && GE::STAGE_COL) ? GE::COL_STAGE_SMEM : 0);
    cudaError_t e = set_smem(k_persist<N, PREC, HEAT, TS>, smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_persist<N, PREC, HEAT, TS>, GE::THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    Params Pc = P;
    void* args[] = {&Pc};
    return cudaLaunchCooperativeKernel((const void*)k_persist<N, PREC, HEAT, TS>, dim3(grid), dim3(GE::THREADS), args,
                                       (size_t)smem, st);
}
}  // namespace

#define SHG_CAT_(a, b) a##b
#define SHG_CAT(a, b) SHG_CAT_(a, b)

cudaError_t SHG_CAT(launch_row_, SHG_N)(const Params& P, int mode, int n, int hsel, bool prec, int grid,
                                        cudaStream_t st) {
    if (P.scheme == 1) {          // the paper's ordering: hi+lo constants only, full-step tables
        if (mode == ROW_FIRST) return launch_row_paper_t<ROW_FIRST>(P, n, grid, st);
        if (mode == ROW_MID) return launch_row_paper_t<ROW_MID>(P, n, grid, st);
        return launch_row_paper_t<ROW_FINAL>(P, n, grid, st);
    }
    if (prec) {
        if (mode == ROW_FIRST) return launch_row_t<ROW_FIRST, true>(P, n, hsel, grid, st);
        if (mode == ROW_MID) return P.Q ? launch_row_t<ROW_MID, true, true>(P, n, hsel, grid, st)
                                        : launch_row_t<ROW_MID, true>(P, n, hsel, grid, st);
        return launch_row_t<ROW_FINAL, true>(P, n, hsel, grid, st);
    } else {
        if (mode == ROW_FIRST) return launch_row_t<ROW_FIRST, false>(P, n, hsel, grid, st);
        if (mode == ROW_MID) return P.Q ? launch_row_t<ROW_MID, false, true>(P, n, hsel, grid, st)
                                        : launch_row_t<ROW_MID, false>(P, n, hsel, grid, st);
        return launch_row_t<ROW_FINAL, false>(P, n, hsel, grid, st);
    }
}

cudaError_t SHG_CAT(launch_col_, SHG_N)(const Params& P, int hsel, bool prec, int grid, cudaStream_t st) {
    return prec ? launch_col_t<true>(P, hsel, grid, st) : launch_col_t<false>(P, hsel, grid, st);
}

cudaError_t SHG_CAT(launch_persist_, SHG_N)(const Params& P, bool prec, int grid, cudaStream_t st) {
    if (P.scheme == 1) {
        const int smem = GE::CTA_SMEM;
        cudaError_t e = set_smem(k_persist_paper<N, true>, smem);
        if (e != cudaSuccess) return e;
        Params Pc = P;
        void* args[] = {&Pc};
        return cudaLaunchCooperativeKernel((const void*)k_persist_paper<N, true>, dim3(grid), dim3(GE::THREADS), args,
                                           (size_t)smem, st);
    }
    if (P.flat_rows) {
        const int smem = GE::CTA_SMEM;
        const void* kf = prec ? (const void*)k_persist_flat<N, true> : (const void*)k_persist_flat<N, false>;
        cudaError_t e = cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        Params Pc = P;
        void* args[] = {&Pc};
        return cudaLaunchCooperativeKernel(kf, dim3(grid), dim3(GE::THREADS), args, (size_t)smem, st);
    }
    if (P.pipeline) {
        const int smem = GE::PIPE_SMEM_STG;
        const void* kf = prec ? (const void*)k_persist_pipe<N, true> : (const void*)k_persist_pipe<N, false>;
        cudaError_t e = cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        Params Pc = P;
        void* args[] = {&Pc};
        return cudaLaunchCooperativeKernel(kf, dim3(grid), dim3(GE::THREADS), args, (size_t)smem, st);
    }
    if (P.Q) return prec ? launch_persist_t<true, true>(P, grid, st) : launch_persist_t<false, true>(P, grid, st);
    if (P.tab_smem && prec) return launch_persist_t<true, false, true>(P, grid, st);
    return prec ? launch_persist_t<true, false>(P, grid, st) : launch_persist_t<false, false>(P, grid, st);
}

#if SHG_N <= 128
namespace {
// One cluster of C CTAs per member (k_cluster).  max_clusters (if not null) receives how many such clusters the
// device can hold at once; launch = false only queries.
template <int C>
cudaError_t launch_cluster_t(const Params& P, bool launch, int* max_clusters, cudaStream_t st) {
    using CG = CGeo<N, C>;
    auto kern = k_cluster<N, C, true>;
    // at least 120 KB: one CTA per SM, so that the CTAs of a cluster never share an SM's pipes
    const int smem = CG::SMEM > 120 * 1024 ? CG::SMEM : 120 * 1024;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    if (C > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(P.batch * C));
    cfg.blockDim = dim3(CG::THREADS);
    cfg.dynamicSmemBytes = (size_t)smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (max_clusters) {
        e = cudaOccupancyMaxActiveClusters(max_clusters, kern, &cfg);
        if (e != cudaSuccess) return e;
    }
    if (!launch) return cudaSuccess;
    return cudaLaunchKernelEx(&cfg, kern, P);
}
}  // namespace
#endif

cudaError_t SHG_CAT(launch_cluster_, SHG_N)(const Params& P, int csize, bool launch, int* max_clusters,
                                            cudaStream_t st) {
#if SHG_N <= 64
    if (csize == 8) return launch_cluster_t<8>(P, launch, max_clusters, st);
#endif
#if SHG_N <= 128
    if (csize == 16) return launch_cluster_t<16>(P, launch, max_clusters, st);
#endif
    (void)P; (void)launch; (void)max_clusters; (void)st; (void)csize;
    return cudaErrorNotSupported;
}

LaunchInfo SHG_CAT(launch_info_, SHG_N)() {
    LaunchInfo li;
    li.rows_per_item = GE::HG;
    li.cols_per_item = GE::SC;
    li.warps = GE::WARPS;
    li.row_slots = GE::ROW_SLOTS;
    li.col_teams = GE::TEAMS;
    li.team_warps = GE::TW;
    li.fft_r = GE::R;
    li.fft_m = GE::M;
    return li;
}

}  // namespace shg
