// fft_launch.cuh — launch geometry and radix plans of the FFT passes; included by fft_f64.cu / fft_f32.cu, which
// instantiate it for one precision each.
#pragma once
#include <cstring>

#include "fft.cuh"
#include "plan.h"

namespace galb {

// ---------------------------------------------------------------------------------------------
// FFT launchers
// ---------------------------------------------------------------------------------------------
template <typename T, int R1, int R2, int R3, int F>
int launch_row(gal_plan* p, const T* image, const SweepParams* sw, int batch, const int* ext, cudaStream_t st) {
    using G = Geom<T, R1, R2, R3, F>;
    RowParams<T> rp;
    rp.image = image;
    rp.spec = (cx<T>*)p->work;
    rp.tw = (const cx<T>*)p->tw;
    rp.N = p->nxy;
    rp.rows_total = batch * p->nxy;
    rp.ext = ext;
    rp.pf_blocks = 0;
    if (sw) rp.sweep = *sw; else memset(&rp.sweep, 0, sizeof(rp.sweep));
    const unsigned grid = (unsigned)((rp.rows_total + F - 1) / F);
    if (sw) {
        auto k = row_pass_kernel<T, R1, R2, R3, F, true>;
        int rc = set_smem(p, k, G::SMEM); if (rc) return rc;
        GAL_CUDA(p, launch_chain(k, dim3(grid), dim3(G::NT), G::SMEM, st, rp));
    } else {
        auto k = row_pass_kernel<T, R1, R2, R3, F, false>;
        int rc = set_smem(p, k, G::SMEM); if (rc) return rc;
        rp.pf_blocks = resident_ctas(p, k, G::NT, G::SMEM);
        GAL_CUDA(p, launch_chain(k, dim3(grid), dim3(G::NT), G::SMEM, st, rp));
    }
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    if (p->tmark(2, st)) return GAL_ERR_CUDA;
    return GAL_OK;
}

// Row pass with lane-interleaved rows and the register untangle (fft.cuh: row_pipe_kernel).  tma: persistent grid,
// one CTA per SM, NG groups and a ring of NS slots; otherwise one row block per CTA and plain loads (or the sweep).
template <typename T, int R1, int R2, int R3, int F, int NG, int NS>
int launch_row_pipe(gal_plan* p, const T* image, const SweepParams* sw, int batch, const int* ext, bool tma, cudaStream_t st) {
    using G = RowGeom<T, R1, R2, R3, F>;
    static_assert(NS >= NG, "one slot per group at least");
    RowParams<T> rp;
    rp.image = image;
    rp.spec = (cx<T>*)p->work;
    rp.tw = (const cx<T>*)p->tw;
    rp.N = p->nxy;
    rp.rows_total = batch * p->nxy;
    rp.ext = ext;
    rp.pf_blocks = 0;
    if (sw) rp.sweep = *sw; else memset(&rp.sweep, 0, sizeof(rp.sweep));
    const long long nblk = rp.rows_total / F;
    if (!sw && tma) {
        const unsigned grid = (unsigned)(nblk < p->sm_count ? nblk : p->sm_count);
        const size_t smem = (size_t)NS * G::SLOT_BYTES + 16 * NS;
        auto k = row_pipe_kernel<T, R1, R2, R3, F, NG, NS, ROW_TMA>;
        int rc = set_smem(p, k, smem); if (rc) return rc;
        GAL_CUDA(p, launch_chain(k, dim3(grid), dim3(G::GT * NG + 32), smem, st, rp));
    } else {
        const size_t smem = (size_t)G::SLOT_BYTES;
        if (sw) return GAL_ERR_UNSUPPORTED;          // *Profile calls take the plain kernel's sweep loader
        auto k = row_pipe_kernel<T, R1, R2, R3, F, 1, 1, ROW_DIRECT>;
        int rc = set_smem(p, k, smem); if (rc) return rc;
        rp.pf_blocks = resident_ctas(p, k, G::GT, smem);
        GAL_CUDA(p, launch_chain(k, dim3((unsigned)nblk), dim3(G::GT), smem, st, rp));
    }
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    if (p->tmark(2, st)) return GAL_ERR_CUDA;
    return GAL_OK;
}

template <typename T, int R1, int R2, int R3, int F>
int launch_col(gal_plan* p, int batch, const int* ext, cudaStream_t st) {
    using G = Geom<T, R1, R2, R3, F>;
    ColParams<T> cp;
    cp.work = (const cx<T>*)p->work;
    cp.pair = (NodePair<T>*)p->spec;
    cp.tw = (const cx<T>*)p->tw;
    cp.N = p->nxy;
    cp.cols_total = (long long)batch * (p->nxy / 2 + 1);
    cp.ext = ext;
    const unsigned grid = (unsigned)((cp.cols_total + F - 1) / F);
    auto k = col_pass_kernel<T, R1, R2, R3, F>;
    int rc = set_smem(p, k, G::SMEM); if (rc) return rc;
    cp.pf_groups = resident_ctas(p, k, G::NT, G::SMEM);
    GAL_CUDA(p, launch_chain(k, dim3(grid), dim3(G::NT), G::SMEM, st, cp));
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

template <typename T, int R1, int R2, int R3>
int launch_col_x2(gal_plan* p, int batch, const int* ext, cudaStream_t st) {
    using G = Geom<T, R1, R2, R3, 2>;
    ColParams<T> cp;
    cp.work = (const cx<T>*)p->work;
    cp.pair = (NodePair<T>*)p->spec;
    cp.tw = (const cx<T>*)p->tw;
    cp.N = p->nxy;
    cp.cols_total = (long long)batch * (p->nxy / 2 + 1);
    cp.ext = ext;
    cp.pf_groups = 0;
    auto k = col_pass_x2_kernel<T, R1, R2, R3>;
    int rc = set_smem(p, k, G::SMEM); if (rc) return rc;
    GAL_CUDA(p, launch_chain(k, dim3((unsigned)cp.cols_total), dim3(G::NT), G::SMEM, st, cp));
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

// nxy = 16384: row pass as two interleaved transforms, column transform four-step through global memory.
template <typename T>
int launch_fft_16384(gal_plan* p, const T* image, const SweepParams* sw, int batch, const int* ext, cudaStream_t st) {
    using GR = Geom<T, 16, 16, 16, 2>;
    using GC = Geom<T, 16, 16, 16, 1>;
    RowParams<T> rp;
    rp.image = image; rp.spec = (cx<T>*)p->work; rp.tw = (const cx<T>*)p->tw; rp.N = p->nxy;
    rp.rows_total = batch * p->nxy; rp.ext = ext; rp.pf_blocks = 0;
    if (sw) rp.sweep = *sw; else memset(&rp.sweep, 0, sizeof(rp.sweep));
    int rc;
    const bool one_cta = p->row_x2_one_cta;                  // GAL_OPT_ROW_X2_ONE_CTA: the one-CTA-per-row form
    if (!one_cta) {
        // a cluster of two CTAs per row (fft.cuh: row_pass_c2_kernel)
        const unsigned grid = 2u * (unsigned)rp.rows_total;
        if (sw) {
            auto k = row_pass_c2_kernel<T, 16, 16, 16, true>;
            if ((rc = set_smem(p, k, GC::SMEM))) return rc;
            GAL_CUDA(p, launch_chain_cluster(k, dim3(grid), dim3(GC::NT), GC::SMEM, 2u, st, rp));
        } else {
            auto k = row_pass_c2_kernel<T, 16, 16, 16, false>;
            if ((rc = set_smem(p, k, GC::SMEM))) return rc;
            rp.pf_blocks = resident_ctas(p, k, GC::NT, GC::SMEM) / 2;        // (in rows)
            GAL_CUDA(p, launch_chain_cluster(k, dim3(grid), dim3(GC::NT), GC::SMEM, 2u, st, rp));
        }
    } else if (sw) {
        auto k = row_pass_x2_kernel<T, 16, 16, 16, true>;
        if ((rc = set_smem(p, k, GR::SMEM))) return rc;
        GAL_CUDA(p, launch_chain(k, dim3((unsigned)rp.rows_total), dim3(GR::NT), GR::SMEM, st, rp));
    } else {
        auto k = row_pass_x2_kernel<T, 16, 16, 16, false>;
        if ((rc = set_smem(p, k, GR::SMEM))) return rc;
        rp.pf_blocks = resident_ctas(p, k, GR::NT, GR::SMEM);
        GAL_CUDA(p, launch_chain(k, dim3((unsigned)rp.rows_total), dim3(GR::NT), GR::SMEM, st, rp));
    }
    p->launches++;
    if (p->tmark(2, st)) return GAL_ERR_CUDA;
    ColParams<T> cp;
    cp.work = (const cx<T>*)p->work; cp.pair = (NodePair<T>*)p->spec; cp.tw = (const cx<T>*)p->tw; cp.N = p->nxy;
    cp.cols_total = (long long)batch * (p->nxy / 2 + 1); cp.ext = ext; cp.pf_groups = 0;
    auto ks = col_sub_kernel<T, 16, 16, 16>;
    if ((rc = set_smem(p, ks, GC::SMEM))) return rc;
    GAL_CUDA(p, launch_chain(ks, dim3((unsigned)(4 * cp.cols_total)), dim3(GC::NT), GC::SMEM, st, cp, (cx<T>*)p->work));
    GAL_CUDA(p, launch_chain(col_comb4_kernel<T>, dim3(4, (unsigned)cp.cols_total), dim3(256), 0, st, cp));
    p->launches += 2;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

// Groups per CTA and ring slots of the pipelined row pass: fp64 slots are 66 KB (two groups, three slots);
// fp32 slots are half that (three groups, five slots).
#ifndef GAL_ROW_NG64
#define GAL_ROW_NG64 2
#endif
#ifndef GAL_ROW_NS64
#define GAL_ROW_NS64 3
#endif
#ifndef GAL_ROW_NG32
#define GAL_ROW_NG32 3
#endif
#ifndef GAL_ROW_NS32
#define GAL_ROW_NS32 5
#endif
template <typename T> struct RowPipeCfg;
// default_mode: which row kernel a size takes when GAL_ROW_PIPE does not say (measured on B200):
// 0 = plain kernel, 1 = lane-interleaved rows + register untangle with plain loads, 2 = its persistent TMA-ring form.
template <> struct RowPipeCfg<double> {
    static constexpr int NG = GAL_ROW_NG64, NS = GAL_ROW_NS64;
    static int default_mode(int nxy) { return nxy >= 2048 ? 1 : 0; }   // (2048: as fast as the plain kernel, and the same arithmetic as its one-row form)
};
template <> struct RowPipeCfg<float> {
    static constexpr int NG = GAL_ROW_NG32, NS = GAL_ROW_NS32;
    static int default_mode(int nxy) { return nxy >= 2048 ? 2 : 0; }
};

// Radix plans.  Row FFT length is nxy/2, column FFT length is nxy.
template <typename T>
int fft2(gal_plan* p, const T* image, const SweepParams* sw, int batch, const int* ext, cudaStream_t st) {
    int rc;
    switch (p->nxy) {
#define GAL_FFT_CASE(NXY, ROW, COL)                                         \
    case NXY:                                                               \
        rc = launch_row<T, ROW>(p, image, sw, batch, ext, st); if (rc) return rc; \
        return launch_col<T, COL>(p, batch, ext, st);
#define RR(...) __VA_ARGS__
        GAL_FFT_CASE(8, RR(4, 1, 1, 8), RR(8, 1, 1, 8))
        GAL_FFT_CASE(16, RR(8, 1, 1, 16), RR(16, 1, 1, 16))
        GAL_FFT_CASE(32, RR(16, 1, 1, 16), RR(8, 4, 1, 16))
        GAL_FFT_CASE(64, RR(8, 4, 1, 16), RR(8, 8, 1, 16))
        GAL_FFT_CASE(128, RR(8, 8, 1, 16), RR(16, 8, 1, 16))
        GAL_FFT_CASE(256, RR(16, 8, 1, 16), RR(16, 16, 1, 8))
        GAL_FFT_CASE(512, RR(16, 16, 1, 8), RR(8, 8, 8, 4))
        // nxy >= 1024: the pipelined row pass (row_mode 0 keeps the plain one, for comparison)
#define GAL_FFT_CASE_PIPE(NXY, ROW, PIPE, COL)                                   \
    case NXY: {                                                                  \
        const int mode = sw ? 0 : (p->row_mode >= 0 ? p->row_mode : RowPipeCfg<T>::default_mode(NXY)); \
        rc = mode ? launch_row_pipe<T, PIPE, RowPipeCfg<T>::NG, RowPipeCfg<T>::NS>(p, image, sw, batch, ext, mode == 2, st) \
                  : launch_row<T, ROW>(p, image, sw, batch, ext, st);            \
        if (rc) return rc;                                                       \
        return launch_col<T, COL>(p, batch, ext, st);                            \
    }
        case 1024: {
            const int mode = sw ? 0 : (p->row_mode >= 0 ? p->row_mode : RowPipeCfg<T>::default_mode(1024));
            // rows: eight per CTA when the batch fills the GPU several times over (cfg 4: 417 -> 406 us), else four
            const bool many = (long long)batch * 1024 / 8 >= 4LL * p->sm_count;
            rc = mode ? launch_row_pipe<T, 16, 8, 4, 8, RowPipeCfg<T>::NG, RowPipeCfg<T>::NS>(p, image, sw, batch, ext, mode == 2, st)
                      : many ? launch_row<T, 8, 8, 8, 8>(p, image, sw, batch, ext, st)
                             : launch_row<T, 8, 8, 8, 4>(p, image, sw, batch, ext, st);
            if (rc) return rc;
            // columns: two per CTA (128 threads, five CTAs per SM) instead of four: cfg 4 column pass 422 -> 357 us
            return launch_col<T, 16, 8, 8, 2>(p, batch, ext, st);
        }
        case 2048: {
            int mode = sw ? 0 : (p->row_mode >= 0 ? p->row_mode : RowPipeCfg<T>::default_mode(2048));
            // as at 4096 (below): one row per CTA where the plan expects a pruned extent (cfg 2: row pass 20.8 -> 18.7 us)
            if (mode == 1 && p->row_small && sizeof(T) == 8) mode = 3;
            if (mode == 3) rc = launch_row_pipe<T, 16, 8, 8, 1, 1, 1>(p, image, sw, batch, ext, false, st);
            else if (mode) rc = launch_row_pipe<T, 16, 8, 8, 4, RowPipeCfg<T>::NG, RowPipeCfg<T>::NS>(p, image, sw, batch, ext, mode == 2, st);
            else rc = launch_row<T, 16, 8, 8, 4>(p, image, sw, batch, ext, st);
            if (rc) return rc;
            return launch_col<T, 16, 16, 8, 2>(p, batch, ext, st);
        }
#undef GAL_FFT_CASE_PIPE
        case 4096: {
            int mode = sw ? 0 : (p->row_mode >= 0 ? p->row_mode : RowPipeCfg<T>::default_mode(4096));
            // A transform pruned to a part of the half plane leaves a row-transformed image of a few tens of MB,
            // which stays in the L2: there ONE row per CTA (barriers over four warps instead of eight, a tail half
            // as long; 16-byte stores that the L2 merges) is faster, 46.5 against 51.3 us at cfg 3.  Written out to
            // HBM (whole plane) the half-sector stores cost a factor of two (147 against 68 us), so the choice
            // follows the extent the plan expects (plan.h row_small).  Mode 3 forces it (diagnostic).
            if (mode == 1 && p->row_small && sizeof(T) == 8) mode = 3;
            if (mode == 3) rc = launch_row_pipe<T, 16, 16, 8, 1, 1, 1>(p, image, sw, batch, ext, false, st);
            else if (mode) rc = launch_row_pipe<T, 16, 16, 8, 2, RowPipeCfg<T>::NG, RowPipeCfg<T>::NS>(p, image, sw, batch, ext, mode == 2, st);
            else rc = launch_row<T, 16, 16, 8, 2>(p, image, sw, batch, ext, st);
            if (rc) return rc;
            return launch_col<T, 16, 16, 16, 1>(p, batch, ext, st);
        }
        case 8192:      // column length 8192 = 2 x 4096: two interleaved transforms + one radix-2 combination
            rc = launch_row<T, 16, 16, 16, 1>(p, image, sw, batch, ext, st); if (rc) return rc;
            return launch_col_x2<T, 16, 16, 16>(p, batch, ext, st);
        case 16384:
            return launch_fft_16384<T>(p, image, sw, batch, ext, st);
#undef RR
#undef GAL_FFT_CASE
        default:
            return GAL_ERR_UNSUPPORTED;
    }
}


template <typename T>
int launch_sweep(gal_plan* p, const SweepParams& sw, T* out, cudaStream_t st) {
    const long long total = (long long)p->nxy * p->nxy;
    long long blocks = (total + 255) / 256;
    if (blocks > p->sm_count * 16) blocks = p->sm_count * 16;
    sweep_kernel<T><<<(unsigned)blocks, 256, 0, st>>>(sw, p->nxy, out);
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

template <typename T>
int launch_transpose(gal_plan* p, T* out, cudaStream_t st) {
    dim3 grid((p->nxy + 31) / 32, (p->nxy / 2 + 1 + 31) / 32), block(32, 8);
    transpose_to_paper_layout_kernel<T><<<grid, block, 0, st>>>((const cx<T>*)p->spec, (cx<T>*)out, p->nxy);
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

#define GAL_INSTANTIATE_FFT(T)                                                                             \
    template int fft2<T>(gal_plan*, const T*, const SweepParams*, int, const int*, cudaStream_t);          \
    template int launch_sweep<T>(gal_plan*, const SweepParams&, T*, cudaStream_t);                         \
    template int launch_transpose<T>(gal_plan*, T*, cudaStream_t);

}  // namespace galb
