// redo.cuh — the conditional second pass of a speculative call (plan.h: speculative extent).
//
// A call on the automatic pruning mode transforms only the part of the half plane the PREVIOUS call's points could
// reach, and its sampler verifies every point against that extent.  When a point lies outside (the uv data grew),
// the result of the first pass is wrong and the sampler's last CTA raises a device flag.  This kernel is launched
// behind every speculative call; it reads the flag and leaves at once in the normal case (one empty launch, about
// 2 us in the chain, instead of a 20 us uv-extent kernel in front of every call).  Otherwise it repeats the whole
// call — row pass, column pass, sampling — on the extent the sampler has just derived from the
// points themselves, as ONE persistent launch with grid barriers between the passes: a rare path, built for
// correctness, not speed.  The row pass is the plain kernel's (fft.cuh: row_block), so a repeated call may differ
// from an unrepeated one in the last bits of the transform, far inside every tolerance.
#pragma once
#include "fft.cuh"
#include "plan.h"
#include "sample.cuh"
#include "sample_launch.cuh"

namespace galb {

struct RedoState {
    unsigned int* flag;    // raised by the sampler of the first pass; cleared here
    unsigned int* bar;     // [2]: grid-barrier counter, exit ticket (both 0 between launches)
};

// Every CTA of the grid is resident (the launcher asks for no more CTAs than fit) and arrives once per barrier.
__device__ __forceinline__ void grid_barrier(unsigned int* bar, unsigned int target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
        while (*reinterpret_cast<volatile unsigned int*>(bar) < target) __nanosleep(128);
        __threadfence();
    }
    __syncthreads();
}

template <typename T, int A1, int A2, int A3, int AF, int B1, int B2, int B3, int BF, bool WRITE_VIS, bool DO_CHI2>
__global__ void __launch_bounds__(256, 1)
redo_kernel(const RowParams<T> rp, const ColParams<T> cp, const SampleParams<T> sp, const RedoState rs) {
    static_assert(Geom<T, A1, A2, A3, AF>::NT == 256 && Geom<T, B1, B2, B3, BF>::NT == 256 && GAL_SAMPLE_NT == 256,
                  "one CTA shape for the three passes");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* smem = reinterpret_cast<cx<T>*>(smem_raw);
    pdl_wait();
    if (*reinterpret_cast<volatile unsigned int*>(rs.flag) == 0u) return;        // the first pass stands
    // ---- row pass (S3 rows)
    const long long nrb = ((long long)rp.rows_total + AF - 1) / AF;
    for (long long vb = blockIdx.x; vb < nrb; vb += gridDim.x) {
        if (vb != (long long)blockIdx.x) __syncthreads();
        row_block<T, A1, A2, A3, AF, false>(rp, vb, smem);
    }
    grid_barrier(rs.bar, gridDim.x);
    // ---- column pass (S2, S3 columns, S4)
    const long long ncg = (cp.cols_total + BF - 1) / BF;
    for (long long g = blockIdx.x; g < ncg; g += gridDim.x) {
        if (g != (long long)blockIdx.x) __syncthreads();
        col_block<T, B1, B2, B3, BF>(cp, g * BF, smem);
    }
    grid_barrier(rs.bar, 2u * gridDim.x);
    if (blockIdx.x == 0 && threadIdx.x == 0) *rs.flag = 0u;                       // every CTA has read it
    // ---- sampling (S5-S8): plain loads, any alignment
    SampleCtx<T> cx_ = sample_ctx(sp, 0);
    const long long ntiles = (sp.M + SampleGeom<T, DO_CHI2>::TILE - 1) / SampleGeom<T, DO_CHI2>::TILE;
    if (layout_single(sp.ext, sp.N)) {
        for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x)
            sample_tile_plain<T, WRITE_VIS, DO_CHI2, true, false>(sp, cx_, tile, sp.M, 0);
    } else {
        for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x)
            sample_tile_plain<T, WRITE_VIS, DO_CHI2, true, true>(sp, cx_, tile, sp.M, 0);
    }
    sample_finish<T, DO_CHI2>(sp, 0, cx_.acc, cx_.oob, cx_.viol);
    __syncthreads();
    if (threadIdx.x == 0 && atomicAdd(rs.bar + 1, 1u) == gridDim.x - 1u) { rs.bar[0] = 0u; rs.bar[1] = 0u; }   // re-arm
}

template <typename T, int A1, int A2, int A3, int AF, int B1, int B2, int B3, int BF>
int launch_redo_plan(gal_plan* p, const T* image, const CallScalars& cs, const T* u, const T* v, const T* re, const T* im,
                     const T* w, int64_t M, T* vis, double* chi2_pc, double* chi2_tot, cudaStream_t st) {
    using GA = Geom<T, A1, A2, A3, AF>;
    using GB = Geom<T, B1, B2, B3, BF>;
    const int* ext = p->spec_E(p->spec_par ^ 1);
    RowParams<T> rp;
    rp.image = image; rp.spec = (cx<T>*)p->work; rp.tw = (const cx<T>*)p->tw; rp.N = p->nxy;
    rp.rows_total = p->nxy; rp.ext = ext; rp.pf_blocks = 0;
    memset(&rp.sweep, 0, sizeof(rp.sweep));
    ColParams<T> cp;
    cp.work = (const cx<T>*)p->work; cp.pair = (NodePair<T>*)p->spec; cp.tw = (const cx<T>*)p->tw; cp.N = p->nxy;
    cp.cols_total = p->nxy / 2 + 1; cp.ext = ext; cp.pf_groups = 0;
    const int* keep = p->cur_ext;
    p->cur_ext = ext;
    SampleParams<T> sp = make_sample_params<T>(p, cs, u, v, re, im, w, M, vis, chi2_pc, chi2_tot, false);
    p->cur_ext = keep;
    sp.direct = 0; sp.ext_check = nullptr; sp.viol_flag = nullptr;      // (rearm = 0: the first pass has re-armed the next call's state)
    RedoState rs;
    rs.flag = p->spec_redo(); rs.bar = p->spec_bar();
    const size_t smem = GA::SMEM > GB::SMEM ? GA::SMEM : GB::SMEM;
    int rc;
    auto launch = [&](auto k) -> int {
        if ((rc = set_smem(p, k, smem))) return rc;
        auto it = p->resident.find((const void*)k);
        if (it == p->resident.end()) {
            int per_sm = 1;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, 256, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
            p->resident[(const void*)k] = per_sm * p->sm_count;
        }
        int grid = p->resident[(const void*)k];
        if (grid > p->max_gx) grid = p->max_gx;              // (one chi2 partial per CTA)
        GAL_CUDA(p, launch_chain(k, dim3((unsigned)grid), dim3(256), smem, st, rp, cp, sp, rs));
        return GAL_OK;
    };
    if (vis) rc = launch(redo_kernel<T, A1, A2, A3, AF, B1, B2, B3, BF, true, false>);
    else rc = launch(redo_kernel<T, A1, A2, A3, AF, B1, B2, B3, BF, false, true>);
    if (rc) return rc;
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

template <typename T>
int launch_redo(gal_plan* p, const T* image, const CallScalars& cs, const T* u, const T* v, const T* re, const T* im, const T* w,
                int64_t M, T* vis, double* chi2_pc, double* chi2_tot, cudaStream_t st) {
    switch (p->nxy) {            // the sizes run_call speculates at; the radix plans of fft_launch.cuh's plain kernels
        case 2048: return launch_redo_plan<T, 16, 8, 8, 4, 16, 16, 8, 2>(p, image, cs, u, v, re, im, w, M, vis, chi2_pc, chi2_tot, st);
        case 4096: return launch_redo_plan<T, 16, 16, 8, 2, 16, 16, 16, 1>(p, image, cs, u, v, re, im, w, M, vis, chi2_pc, chi2_tot, st);
        default: return GAL_ERR_UNSUPPORTED;
    }
}

#define GAL_INSTANTIATE_REDO(T)                                                                                          \
    template int launch_redo<T>(gal_plan*, const T*, const CallScalars&, const T*, const T*, const T*, const T*, const T*, \
                                int64_t, T*, double*, double*, cudaStream_t);

}  // namespace galb
