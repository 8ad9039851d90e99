// redo.cuh — the conditional second pass of a speculative call (plan.h: speculative extent).
//
// A call on the automatic pruning mode transforms only the part of the half plane the PREVIOUS call's points could
// reach, and its sampler verifies every point against that extent.  When a point lies outside (the uv data grew),
// the result of the first pass is wrong and the sampler's last CTA raises a device flag.  This kernel is launched
// behind every speculative call; it reads the flag and leaves at once in the normal case (one empty launch, about
// 2 us in the chain, instead of a 20 us uv-extent kernel in front of every call).  Otherwise it repeats the whole
// call — row pass, column pass, sampling — on the extent the sampler has just derived from the
// points themselves, as ONE persistent launch whose passes are separated by completion counters (below; it cannot
// dead-lock whatever else runs on the GPU): a rare path, built for correctness, not speed.  The row pass is the plain kernel's (fft.cuh: row_block), so a repeated call may differ
// from an unrepeated one in the last bits of the transform, far inside every tolerance.
#pragma once
#include "fft.cuh"
#include "plan.h"
#include "sample.cuh"
#include "sample_launch.cuh"

namespace galb {

struct RedoState {
    unsigned int* flag;    // raised by the sampler of the first pass; cleared here by the last CTA to leave
    unsigned int* ctr;     // [5]: row blocks claimed, row blocks done, column groups claimed, column groups done, exit ticket (all 0 between launches)
};

// No CTA of this kernel ever waits for another CTA to ARRIVE — only for work that some CTA has already claimed, and a
// CTA that has claimed work is running and will finish it.  So the kernel needs no co-residency guarantee: with other
// work on the GPU (a second plan repeating a call on another stream, each grid wanting every SM; an MPS neighbour; a
// partition smaller than the occupancy query saw) the CTAs that do get placed transform everything, and a CTA placed
// late finds nothing left to claim, both counters complete, and goes straight to its share of the sampling.  (A grid
// barrier that counts arrivals would spin for ever there; a cooperative launch avoids that too, but costs 7 us per
// call even when the kernel leaves at once — measured: cfg 3 119.5 -> 127.1 us.)
//   claim: thread 0 takes the next item of a pass from an atomic counter and hands it to the CTA.
//   done:  after the item's last store, one release per CTA on the pass's completion counter.
//   wait:  a pass may only be read once its completion counter has reached the number of items.
__device__ __forceinline__ long long redo_claim(unsigned int* ctr, long long* slot) {
    __syncthreads();                                         // (the slot and the shared tile of the item before are free)
    if (threadIdx.x == 0) *slot = (long long)atomicAdd(ctr, 1u);
    __syncthreads();
    return *slot;
}
__device__ __forceinline__ void redo_done(unsigned int* done) {
    __syncthreads();
    if (threadIdx.x == 0) { __threadfence(); atomicAdd(done, 1u); }
}
__device__ __forceinline__ void redo_wait(unsigned int* done, unsigned int target) {
    if (threadIdx.x == 0) {
        while (*reinterpret_cast<volatile unsigned int*>(done) < target) __nanosleep(128);
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
    __shared__ long long slot;
    cx<T>* smem = reinterpret_cast<cx<T>*>(smem_raw);
    pdl_wait();
    if (*reinterpret_cast<volatile unsigned int*>(rs.flag) == 0u) return;        // the first pass stands
    // ---- row pass (S3 rows)
    const long long nrb = ((long long)rp.rows_total + AF - 1) / AF;
    for (long long vb = redo_claim(rs.ctr, &slot); vb < nrb; vb = redo_claim(rs.ctr, &slot)) {
        row_block<T, A1, A2, A3, AF, false>(rp, vb, smem);
        redo_done(rs.ctr + 1);
    }
    redo_wait(rs.ctr + 1, (unsigned int)nrb);
    // ---- column pass (S2, S3 columns, S4)
    const long long ncg = (cp.cols_total + BF - 1) / BF;
    for (long long g = redo_claim(rs.ctr + 2, &slot); g < ncg; g = redo_claim(rs.ctr + 2, &slot)) {
        col_block<T, B1, B2, B3, BF>(cp, g * BF, smem);
        redo_done(rs.ctr + 3);
    }
    redo_wait(rs.ctr + 3, (unsigned int)ncg);
    // ---- sampling (S5-S8): plain loads, any alignment.  Tiles are assigned STATICALLY (blockIdx.x, + gridDim.x, ...):
    // nothing waits for this pass, and the chi2 partial of a CTA must not depend on the order the CTAs happened to run in.
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
    // the last CTA to leave re-arms the counters and lowers the flag (every CTA has read it by then)
    if (threadIdx.x == 0 && atomicAdd(rs.ctr + 4, 1u) == gridDim.x - 1u) {
        rs.ctr[0] = 0u; rs.ctr[1] = 0u; rs.ctr[2] = 0u; rs.ctr[3] = 0u; rs.ctr[4] = 0u;
        *rs.flag = 0u;
    }
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
    rs.flag = p->spec_redo(); rs.ctr = p->spec_ctr();
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
        if (grid > p->max_gx) grid = p->max_gx;              // (one chi2 partial per CTA; the size is a matter of speed only)
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
