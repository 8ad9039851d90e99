// sample_launch.cuh — launch geometry of the per-point kernels; included by sample_f64.cu / sample_f32.cu.
#pragma once
#include <cstdlib>
#include "plan.h"
#include "sample.cuh"
#include "sort.cuh"
#include "hankel.cuh"

namespace galb {

template <typename T>
int launch_extent(gal_plan* p, int C, const CallScalars& cs, const T* u, const T* v, int64_t M, cudaStream_t st) {
    ExtentParams ep;
    ep.N = p->nxy;
    ep.total = (long long)C * M;
    ep.ix = cs.ix;
    ep.ext = p->ext;
    long long blocks = (ep.total + 1023) / 1024;
    const long long cap = (long long)p->sm_count * 4;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    GAL_CUDA(p, launch_chain(uv_extent_kernel<T>, dim3((unsigned)blocks), dim3(256), 0, st, ep, u, v));
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

inline bool aligned16(const void* q) { return ((uintptr_t)q & 15u) == 0; }

template <typename T, bool WRITE_VIS, bool DO_CHI2>
int launch_sample_kernel(gal_plan* p, const SampleParams<T>& sp, dim3 grid, bool tma, cudaStream_t st) {
    using G = SampleGeom<T, DO_CHI2>;
    if (tma) {
        auto k = sample_kernel_tma<T, WRITE_VIS, DO_CHI2>;
        int rc = set_smem(p, k, G::SMEM); if (rc) return rc;
        GAL_CUDA(p, launch_chain(k, grid, dim3(G::NT_TMA), G::SMEM, st, sp));
    } else {
        GAL_CUDA(p, launch_chain(sample_kernel_plain<T, WRITE_VIS, DO_CHI2>, grid, dim3(G::NT), 0, st, sp));
    }
    return GAL_OK;
}

// The parameter block of a sampling launch on the plan's current call state (shared with the conditional second
// pass, redo.cuh).
template <typename T>
SampleParams<T> make_sample_params(gal_plan* p, const CallScalars& cs, const T* u, const T* v, const T* re, const T* im, const T* w,
                                   int64_t M, T* vis, double* chi2_pc, double* chi2_tot, bool last) {
    SampleParams<T> sp;
    sp.spec = (const NodePair<T>*)p->spec;
    sp.N = p->nxy;
    sp.M = M;
    sp.u = u; sp.v = v; sp.re_obs = re; sp.im_obs = im; sp.w = w; sp.vis = vis;
    sp.ix = cs.ix;
    sp.amp = cs.amp; sp.accumulate = cs.accumulate;
    sp.dRA_turns = cs.dRA_turns; sp.dDec_turns = cs.dDec_turns; sp.has_phase = cs.has_phase;
    sp.partials = p->partials;
    sp.tickets = p->tickets;
    sp.chi2_per_channel = chi2_pc;
    sp.chi2_total = chi2_tot;
    sp.oob = p->oob;
    sp.done = (unsigned int*)((char*)p->oob + 20);
    sp.next_state = (unsigned long long*)((char*)p->call_state + 32 * (p->cur ^ 1));
    sp.viol = (unsigned long long*)((char*)p->oob + 24);
    sp.ext = p->cur_ext;
    sp.rearm = last;
    sp.direct = p->last_obs ? 1 : 0;
    sp.shared_spec = p->shared_spec ? 1 : 0;
    sp.ext_check = (p->last_bound && !p->last_obs && p->b_ext[0] < p->nxy / 2) ? p->b_ext_dev : nullptr;
    sp.viol_flag = p->viol_dev;
    sp.ext_hint = p->viol_dev + 1;
    sp.r2max = nullptr; sp.spec_out = nullptr; sp.redo = p->spec_redo(); sp.used_ext = p->spec_used();
    return sp;
}

template <typename T>
int launch_sample(gal_plan* p, int C, const CallScalars& cs, const T* u, const T* v, const T* re, const T* im,
                  const T* w, int64_t M, T* vis, double* chi2_pc, double* chi2_tot, bool last, cudaStream_t st) {
    const bool do_chi2 = (vis == nullptr);
    if (M == 0) {
        if (chi2_pc) GAL_CUDA(p, cudaMemsetAsync(chi2_pc, 0, sizeof(double) * C, st));
        if (chi2_tot) GAL_CUDA(p, cudaMemsetAsync(chi2_tot, 0, sizeof(double), st));
        return GAL_OK;
    }
    SampleParams<T> sp = make_sample_params<T>(p, cs, u, v, re, im, w, M, vis, chi2_pc, chi2_tot, last);
    // speculative extent (plan.h spec_mode): 1 = derive the next call's extent, 2 = verify this call's and derive
    const bool spec = p->spec_mode == 1 || p->spec_mode == 2;
    if (spec) {
        sp.r2max = (unsigned long long*)p->spec_state;
        sp.spec_out = p->spec_E(p->spec_par ^ 1);
        if (p->spec_mode == 2) { sp.ext_check = p->cur_ext; sp.viol_flag = nullptr; }
    }
    // one CTA works through tiles blockIdx.x, blockIdx.x + gridDim.x, ...: a whole number of CTAs per SM
    const int tile = SampleGeom<T, true>::TILE;
    const long long ntiles = (M + tile - 1) / tile;
    long long cap = (long long)p->sm_count * GAL_SAMPLE_MINB;
    // batched: CTAs are placed channel by channel (blockIdx.x fastest); a twelfth of the resident CTAs per
    // channel keeps about twelve channels' spectra (not dozens) competing for the L2 at any time and gives every
    // CTA enough tiles to amortise its prologue and reduction (measured at cfg 4, bound observations: 4: 437,
    // 8: 396, 12: 384, 16: 385 us)
    const int conc = p->batch_conc;                      // channels in flight (GAL_OPT_BATCH_CONC)
    if (C > 1) cap = (cap + (C < conc ? C : conc) - 1) / (C < conc ? C : conc);
    if (cap > p->max_gx) cap = p->max_gx;
    long long gx = ntiles < cap ? ntiles : cap;
    if (gx < 1) gx = 1;
    dim3 grid((unsigned)gx, (unsigned)C);
    // the TMA path needs 16-byte aligned tiles in every channel (and a du fit for the division shortcut)
    bool tma = !cs.ix.du_exact_div && aligned16(u) && aligned16(v) && (C == 1 || ((size_t)M * sizeof(T)) % 16 == 0);
    if (do_chi2) tma = tma && aligned16(re) && aligned16(im) && aligned16(w);
    int rc;
    if (spec) {                                   // (run_call only speculates on aligned arrays: the TMA kernel)
        using G = SampleGeom<T, true>;
        if (!tma) return GAL_ERR_INVALID_ARGUMENT;
        if (do_chi2) {
            auto k = sample_kernel_tma<T, false, true, true>;
            if ((rc = set_smem(p, k, SampleGeom<T, true>::SMEM))) return rc;
            GAL_CUDA(p, launch_chain(k, grid, dim3(G::NT_TMA), SampleGeom<T, true>::SMEM, st, sp));
        } else {
            auto k = sample_kernel_tma<T, true, false, true>;
            if ((rc = set_smem(p, k, SampleGeom<T, false>::SMEM))) return rc;
            GAL_CUDA(p, launch_chain(k, grid, dim3(G::NT_TMA), SampleGeom<T, false>::SMEM, st, sp));
        }
        rc = GAL_OK;
    } else {
        rc = do_chi2 ? launch_sample_kernel<T, false, true>(p, sp, grid, tma, st)
                     : launch_sample_kernel<T, true, false>(p, sp, grid, tma, st);
    }
    if (rc) return rc;
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    p->next_armed = last;                 // the last CTA of a call's last launch re-arms the other copy of the call state
    return GAL_OK;
}

template <typename T>
int launch_uv_radius(gal_plan* p, const T* u, const T* v, long long total, cudaStream_t st) {
    long long blocks = (total + 1023) / 1024;
    if (blocks > (long long)p->sm_count * 8) blocks = (long long)p->sm_count * 8;
    uv_radius_kernel<T><<<(unsigned)blocks, 256, 0, st>>>(u, v, total, p->b_r2);
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

// gal_plan_bind_obs: Morton keys, three stable 8-bit radix passes over (key, index), gather (sort.cuh).  Bind-time
// only: temporary buffers are allocated and freed here and the stream is synchronised.
template <typename T>
int launch_bind_sort(gal_plan* p, const T* u, const T* v, const T* re, const T* im, const T* w, int64_t M, int C,
                     double rmax, T* dst, cudaStream_t st) {
    const int ntiles = (int)((M + SORT_TILE - 1) / SORT_TILE);
    unsigned int *key[2] = {nullptr, nullptr}, *idx[2] = {nullptr, nullptr}, *hist = nullptr;
    auto release = [&]() { cudaFree(key[0]); cudaFree(key[1]); cudaFree(idx[0]); cudaFree(idx[1]); cudaFree(hist); };
    const size_t nb = sizeof(unsigned int) * (size_t)M;
    cudaError_t e = cudaSuccess;
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) { e = cudaMalloc(&key[i], nb); if (e == cudaSuccess) e = cudaMalloc(&idx[i], nb); }
    if (e == cudaSuccess) e = cudaMalloc(&hist, sizeof(unsigned int) * 256 * (size_t)ntiles);
    if (e != cudaSuccess) { release(); p->last_cuda = (int)e; return GAL_ERR_ALLOC; }
    const size_t sc_smem = sizeof(unsigned short) * 256 * SORT_STRIDE;
    e = cudaFuncSetAttribute(radix_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sc_smem);
    long long gb = (M + 255) / 256;
    if (gb > (long long)p->sm_count * 8) gb = (long long)p->sm_count * 8;
    const double inv_rmax = rmax > 0 ? 1.0 / rmax : 0.0;
    for (int c = 0; c < C && e == cudaSuccess; ++c) {
        const size_t o = (size_t)c * M;
        uv_key_kernel<T><<<(unsigned)gb, 256, 0, st>>>(u + o, v + o, M, inv_rmax, key[0], idx[0]);
        int cur = 0;
        for (int shift = 0; shift < 24; shift += 8, cur ^= 1) {
            radix_hist_kernel<<<ntiles, SORT_NT, 0, st>>>(key[cur], M, shift, hist, ntiles);
            scan_exclusive_kernel<<<1, 1024, 0, st>>>(hist, 256LL * ntiles);
            radix_scatter_kernel<<<ntiles, SORT_NT, sc_smem, st>>>(key[cur], idx[cur], M, shift, hist, ntiles, key[cur ^ 1],
                                                                    idx[cur ^ 1]);
        }
        T* d = dst + o;
        const size_t plane = (size_t)C * M;
        gather_obs_kernel<T><<<(unsigned)gb, 256, 0, st>>>(idx[cur], M, u + o, v + o, re + o, im + o, w + o, d, d + plane,
                                                           d + 2 * plane, d + 3 * plane, d + 4 * plane);
        p->launches += 11;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    release();
    if (e != cudaSuccess) { p->last_cuda = (int)e; return GAL_ERR_CUDA; }
    return GAL_OK;
}

// Multi-source sampling, one launch per chunk of GAL_MULTI_CHUNK placements (sample.cuh: sample_multi_kernel).
template <typename T>
int launch_sample_multi(gal_plan* p, const IndexScalars& ix, const PlacementSet& ps, const T* u, const T* v, const T* re,
                        const T* im, const T* w, int64_t M, T* vis, bool write_vis, double* chi2, bool last, cudaStream_t st) {
    SampleParams<T> sp = {};
    sp.spec = (const NodePair<T>*)p->spec;
    sp.N = p->nxy; sp.M = M; sp.u = u; sp.v = v; sp.re_obs = re; sp.im_obs = im; sp.w = w; sp.vis = vis; sp.ix = ix;
    sp.partials = p->partials; sp.tickets = p->tickets; sp.chi2_per_channel = chi2; sp.chi2_total = nullptr;
    sp.oob = p->oob; sp.done = (unsigned int*)((char*)p->oob + 20);
    sp.next_state = (unsigned long long*)((char*)p->call_state + 32 * (p->cur ^ 1));
    sp.viol = (unsigned long long*)((char*)p->oob + 24); sp.ext = p->cur_ext; sp.viol_flag = p->viol_dev; sp.rearm = last;
    // as make_sample_params: a bound uv set pruned below the whole plane is verified point by point (a changed set
    // raises GAL_ERR_BINDING_VIOLATED on the next call); the last CTA leaves the row-pass hint for the next call
    sp.ext_check = (p->last_bound && !p->last_obs && p->b_ext[0] < p->nxy / 2) ? p->b_ext_dev : nullptr;
    sp.ext_hint = p->viol_dev + 1;
    long long blocks = (M + 255) / 256;
    const long long cap = (long long)p->sm_count * 6 < p->max_gx ? (long long)p->sm_count * 6 : p->max_gx;
    if (blocks > cap) blocks = cap;
    if (write_vis) GAL_CUDA(p, launch_chain(sample_multi_kernel<T, true, false>, dim3((unsigned)blocks), dim3(256), 0, st, sp, ps));
    else GAL_CUDA(p, launch_chain(sample_multi_kernel<T, false, true>, dim3((unsigned)blocks), dim3(256), 0, st, sp, ps));
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    p->next_armed = last;
    return GAL_OK;
}

// Rotation-invariant extent on the device: radius reduction, then one thread turns it into {kumax, rmin, rmax}.
template <typename T>
int launch_extent_radius(gal_plan* p, const T* u, const T* v, int64_t M, double du, cudaStream_t st) {
    GAL_CUDA(p, cudaMemsetAsync(p->b_r2, 0, 8, st));
    int rc = launch_uv_radius<T>(p, u, v, (long long)M, st);
    if (rc) return rc;
    extent_from_radius_kernel<<<1, 1, 0, st>>>(p->b_r2, du, p->nxy, p->ext);
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

template <typename T>
int launch_sum_channels(gal_plan* p, const double* chi2_pc, int C, double* chi2_tot, cudaStream_t st) {
    GAL_CUDA(p, launch_chain(sum_channels_kernel, dim3(1), dim3(1), 0, st, chi2_pc, C, chi2_tot));
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    return GAL_OK;
}

// Direct Hankel evaluation (hankel.cuh): one warp per point, eight warps per CTA.
template <typename T>
int launch_hankel(gal_plan* p, const SweepParams& sw, const CallScalars& cs, const T* u, const T* v, const T* re, const T* im,
                  const T* w, int64_t M, T* vis, double* chi2, cudaStream_t st) {
    HankelParams h;
    h.I = sw.I; h.nr = sw.nr; h.Rmin = sw.Rmin; h.dR = sw.dR; h.inc_cos = sw.inc_cos;
    h.cos_PA = cs.ix.cos_PA; h.sin_PA = cs.ix.sin_PA; h.dRA_turns = cs.dRA_turns; h.dDec_turns = cs.dDec_turns;
    h.has_phase = cs.has_phase;
    SampleParams<T> sp = {};
    sp.N = p->nxy; sp.M = M; sp.u = u; sp.v = v; sp.re_obs = re; sp.im_obs = im; sp.w = w; sp.vis = vis;
    sp.partials = p->partials; sp.tickets = p->tickets; sp.chi2_per_channel = chi2; sp.chi2_total = nullptr;
    sp.oob = p->oob; sp.done = (unsigned int*)((char*)p->oob + 20);
    sp.next_state = (unsigned long long*)((char*)p->call_state + 32 * (p->cur ^ 1));
    sp.viol = (unsigned long long*)((char*)p->oob + 24); sp.ext_check = nullptr; sp.viol_flag = p->viol_dev; sp.rearm = 1;
    long long blocks = (M + 7) / 8;
    if (blocks > p->max_gx) blocks = p->max_gx;
    if (vis) GAL_CUDA(p, launch_chain(hankel_kernel<T, true, false>, dim3((unsigned)blocks), dim3(256), 0, st, h, sp));
    else GAL_CUDA(p, launch_chain(hankel_kernel<T, false, true>, dim3((unsigned)blocks), dim3(256), 0, st, h, sp));
    p->launches++;
    GAL_CUDA(p, cudaGetLastError());
    p->next_armed = true;
    return GAL_OK;
}

#define GAL_INSTANTIATE_SAMPLE(T)                                                                                      \
    template int launch_extent<T>(gal_plan*, int, const CallScalars&, const T*, const T*, int64_t, cudaStream_t);      \
    template int launch_sample<T>(gal_plan*, int, const CallScalars&, const T*, const T*, const T*, const T*, const T*, \
                                  int64_t, T*, double*, double*, bool, cudaStream_t);                                  \
    template int launch_bind_sort<T>(gal_plan*, const T*, const T*, const T*, const T*, const T*, int64_t, int, double, T*, \
                                     cudaStream_t);                                                                    \
    template int launch_hankel<T>(gal_plan*, const SweepParams&, const CallScalars&, const T*, const T*, const T*, const T*, \
                                  const T*, int64_t, T*, double*, cudaStream_t);                                       \
    template int launch_sample_multi<T>(gal_plan*, const IndexScalars&, const PlacementSet&, const T*, const T*, const T*, \
                                        const T*, const T*, int64_t, T*, bool, double*, bool, cudaStream_t);           \
    template int launch_extent_radius<T>(gal_plan*, const T*, const T*, int64_t, double, cudaStream_t);                \
    template int launch_sum_channels<T>(gal_plan*, const double*, int, double*, cudaStream_t);                         \
    template int launch_uv_radius<T>(gal_plan*, const T*, const T*, long long, cudaStream_t);

}  // namespace galb
