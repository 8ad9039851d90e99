// galario_b200.cu — plan object, kernel dispatch and the C ABI declared in include/galario_b200.h.
// Everything on the path runs in the kernels of fft.cuh and sample.cuh; this file only validates
// arguments, picks the launch geometry and launches on the caller's stream.
#include "../../include/galario_b200.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <set>
#include <vector>

#include "plan.h"

using namespace galb;

extern "C" int gal_plan_unbind_uv(gal_plan* p);
extern "C" int gal_plan_unbind_obs(gal_plan* p);

namespace {

inline bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
inline bool aligned_to(const void* q, size_t n) { return ((uintptr_t)q % n) == 0; }

// ---------------------------------------------------------------------------------------------
// per-call scalars, uv extent, sampling launcher
// ---------------------------------------------------------------------------------------------
// host-side scalars, plain double arithmetic in the listing's order.  The
// phase offsets are kept in turns (the listing's 2 pi factor is applied inside sincospi, exactly).
CallScalars call_scalars(const gal_plan* p, double dxy, double dRA, double dDec, double PA) {
    CallScalars cs;
    IndexScalars& ix = cs.ix;
    ix.du = 1.0 / ((double)p->nxy * dxy);
    ix.rdu = 1.0 / ix.du;
    // Markstein's shortcut needs a divisor whose significand is not all ones
    uint64_t bits; memcpy(&bits, &ix.du, 8);
    ix.du_exact_div = ((bits & 0xFFFFFFFFFFFFFull) == 0xFFFFFFFFFFFFFull) || !std::isnormal(ix.du) || !std::isnormal(ix.rdu);
    ix.cos_PA = std::cos(PA);
    ix.sin_PA = std::sin(PA);
    ix.fH = (double)(p->nxy / 2);
    ix.fHm1 = ix.fH - 1.0;
    ix.fN1 = (double)(p->nxy - 1);
    cs.dRA_turns = dRA * ix.cos_PA - dDec * ix.sin_PA;
    cs.dDec_turns = dRA * ix.sin_PA + dDec * ix.cos_PA;
    cs.has_phase = !(cs.dRA_turns == 0.0 && cs.dDec_turns == 0.0);
    return cs;
}

// Re-arm the per-call device state: out-of-grid counter = 0, uv extent = the cell of the dead slots
// (column 0..1, rows N/2..N/2+1), which the sampler reads with weight 0 for the points past the end.
int reset_call_state(gal_plan* p, cudaStream_t st) {
    p->cur ^= 1;
    p->oob = (unsigned long long*)((char*)p->call_state + 32 * p->cur);
    p->ext = (int*)((char*)p->oob + 8);
    if (!p->next_armed)
        GAL_CUDA(p, cudaMemcpyAsync(p->oob, p->call_init, 32, cudaMemcpyDeviceToDevice, st));
    p->next_armed = false;
    return GAL_OK;
}

// Should this call compute the uv extent and prune the transform?  The extent pass re-reads u and v
// (2 sizeof(T) M bytes per channel); pruning can save up to three passes over the spectrum.
template <typename T>
bool want_prune(const gal_plan* p, int C, int64_t M, int n_spec = 0) {
    if (n_spec <= 0) n_spec = C;                 // spectra transformed by the call (1 for K observation sets of one image)
    if (p->prune_mode == 0 || M <= 0) return false;
    if (p->prune_mode == 2) return true;
    const double ext_bytes = 2.0 * sizeof(T) * (double)M * C;
    const double spec_one = 2.0 * sizeof(T) * (double)(p->nxy / 2 + 1) * p->nxy;
    // a spectrum of a few MB is transformed in a few microseconds out of the L2: the extra launch cannot pay
    // (cfg 0 / 1 / 4: the uv-extent kernel was 15-20 % of the call and mostly found "whole plane")
    if (spec_one < 16e6) return false;
    return ext_bytes <= 0.25 * 3.0 * spec_one * n_spec;
}

// Bound uv set: the extent follows from the radius computed once at bind time, for any PA.  The index of a rotated
// coordinate is at most r_max / du (+ rounding: two cells of margin); rows are symmetric about N/2.  Uploaded once
// per (binding, dxy).
int bound_extent(gal_plan* p, const CallScalars& cs, double dxy, cudaStream_t st) {
    if (p->b_dxy == dxy) return GAL_OK;
    const int H = p->nxy / 2;
    const double imax = p->b_rmax / cs.ix.du;
    int e3[4] = {H, 0, p->nxy - 1, 0};
    if (imax + 3.0 < (double)(H - 1)) {
        const int k = (int)imax + 2;
        e3[0] = k + 1; e3[1] = H - k - 1; e3[2] = H + k + 1;
    }
    GAL_CUDA(p, cudaMemcpyAsync(p->b_ext_dev, e3, sizeof(e3), cudaMemcpyHostToDevice, st));
    GAL_CUDA(p, cudaStreamSynchronize(st));           // e3 is on the stack; once per (binding, dxy)
    p->b_ext[0] = e3[0]; p->b_ext[1] = e3[1]; p->b_ext[2] = e3[2];
    p->b_dxy = dxy;
    return GAL_OK;
}

// Channels per chunk of a batched call.  The kernels of one chunk run back to back (row pass, column pass,
// sampling) on the SAME part of the plan's workspace, so that a chunk's intermediates could stay in the 126 MB L2.
// Measured on B200 at cfg 4 (128 x 1024^2): 1330 us unchunked, 1564 / 1802 / 2205 / 3811 us with 8 / 4 / 2 / 1
// channels per chunk — launches of a few channels are latency-bound (about 10 us per kernel whatever it moves), so
// the default is ONE chunk; GAL_BATCH_CHUNK keeps the experiment reproducible.
int batch_chunk(const gal_plan* p, int C) {
    if (C <= 1 || p->batch_chunk <= 0) return C;
    return p->batch_chunk < C ? p->batch_chunk : C;
}

// One whole call: [uv extent] -> per chunk of channels { row pass -> column pass -> sampling }, with (diagnostic
// mode, gal_plan_timing_enable) a CUDA event after every kernel.
template <typename T>
int run_call(gal_plan* p, const T* image, const SweepParams* sw, int C, double dxy, const T* u, const T* v,
             const T* re, const T* im, const T* w, int64_t M, double dRA, double dDec, double PA, T* vis,
             double* chi2_pc, double* chi2_tot, cudaStream_t st) {
    const CallScalars cs = call_scalars(p, dxy, dRA, dDec, PA);
    p->t_on = p->t_calls < p->t_max_calls;
    int rc;
    if ((rc = reset_call_state(p, st))) return rc;
    if (p->tmark(0, st)) return GAL_ERR_CUDA;
    const int* ext = p->ext_full;
    p->last_pruned = want_prune<T>(p, C, M, p->shared_spec ? 1 : C) && !cs.ix.du_exact_div;   // the extent kernel only has the division shortcut
    p->last_bound = false;
    p->last_obs = false;
    const bool uv_bound = M > 0 && p->b_u == (const void*)u && p->b_v == (const void*)v && p->b_M == M && p->b_C == C;
    if (uv_bound && !vis && p->o_buf && p->o_src[2] == (const void*)re && p->o_src[3] == (const void*)im &&
        p->o_src[4] == (const void*)w) {
        // bound observation set: chi2 does not depend on the order of the points, so sample the plan's private copy,
        // sorted along a space-filling curve of the uv plane (sort.cuh)
        const size_t plane = (size_t)C * M;
        const T* o = (const T*)p->o_buf;
        u = o; v = o + plane; re = o + 2 * plane; im = o + 3 * plane; w = o + 4 * plane;
        p->last_obs = true;
    }
    if (p->prune_mode != 0 && uv_bound) {
        if ((rc = bound_extent(p, cs, dxy, st))) return rc;
        p->last_bound = true;
        p->last_pruned = false;
        ext = p->b_ext_dev;
    }
    // speculative extent (plan.h): possible where this call would otherwise run the uv-extent kernel; an image call on
    // 16-byte aligned arrays (the sampler's TMA form) at a size the conditional second pass is built for
    const bool all16 = aligned_to(u, 16) && aligned_to(v, 16) && (vis || (aligned_to(re, 16) && aligned_to(im, 16) && aligned_to(w, 16)));
    const bool can_spec = p->last_pruned && p->prune_mode == 1 && C == 1 && M > 0 && image && !sw && !p->spec_off && all16 &&
                          (p->nxy == 2048 || p->nxy == 4096) &&
                          (2.0 * sizeof(T) * (double)M >= p->spec_min_bytes);   // (a short extent pass costs no more than the conditional launch)
    const bool speculate = can_spec && p->spec_valid && p->spec_dxy == dxy && p->spec_stream == st;
    p->last_spec = speculate;
    p->spec_mode = speculate ? 2 : (can_spec ? 1 : 0);
    if (speculate) {
        p->last_pruned = false;
        ext = p->spec_E(p->spec_par);
    } else if (p->last_pruned) {
        if ((rc = launch_extent<T>(p, C, cs, u, v, M, st))) return rc;
        ext = p->ext;
    }
    if (p->tmark(1, st)) return GAL_ERR_CUDA;
    p->cur_ext = ext;
    p->row_small = p->last_bound ? p->b_ext[0] < p->nxy / 2
                                 : ((p->last_pruned || speculate) && ((volatile unsigned int*)p->viol_host)[1] == 2u);
    if (M == 0) return launch_sample<T>(p, C, cs, u, v, re, im, w, M, vis, chi2_pc, chi2_tot, true, st);
    const int G = p->shared_spec ? C : batch_chunk(p, C);      // (one image, one transform: nothing to chunk)
    const size_t n2 = (size_t)p->nxy * p->nxy;
    for (int c0 = 0; c0 < C; c0 += G) {
        const int g = C - c0 < G ? C - c0 : G;
        const bool last = c0 + g >= C;
        const size_t o = (size_t)c0 * M;
        if ((rc = fft2<T>(p, image ? image + (p->shared_spec ? 0 : c0 * n2) : nullptr, sw, p->shared_spec ? 1 : g, ext, st))) return rc;
        if (p->tmark(3, st)) return GAL_ERR_CUDA;
        if ((rc = launch_sample<T>(p, g, cs, u + o, v + o, re ? re + o : nullptr, im ? im + o : nullptr, w ? w + o : nullptr, M,
                                   vis ? vis + 2 * o : nullptr, chi2_pc ? chi2_pc + c0 : nullptr, G >= C ? chi2_tot : nullptr, last, st)))
            return rc;
        // speculative call: the conditional second pass (it leaves at once unless the sampler found a point outside)
        if (speculate && (rc = launch_redo<T>(p, image, cs, u, v, re, im, w, M, vis, chi2_pc, chi2_tot, st))) return rc;
        if (p->tmark(4, st)) return GAL_ERR_CUDA;
    }
    if (p->spec_mode != 0) {                   // the sampler has derived (will have, in stream order) the next extent
        p->spec_par ^= 1;
        p->spec_valid = true; p->spec_dxy = dxy; p->spec_stream = st;
        p->spec_mode = 0;
    }
    if (G < C && chi2_tot && (rc = launch_sum_channels<T>(p, chi2_pc, C, chi2_tot, st))) return rc;
    if (p->t_on) { p->t_calls++; p->t_on = false; }
    return GAL_OK;
}

template <typename T> bool prec_ok(const gal_plan* p) { return p && p->bits == (int)(8 * sizeof(T)); }

bool sweep_args(const gal_plan* p, const void* I, int nr, double Rmin, double dR, double dxy, double inc,
                SweepParams* sw) {
    if (!I || nr < 2 || !(dR > 0) || !(dxy > 0) || !std::isfinite(Rmin) || !std::isfinite(inc)) return false;
    const double c = std::cos(inc);
    if (!(std::fabs(inc) < 1.5707963267948966) || !(c > 0)) return false;
    sw->I = I; sw->nr = nr; sw->Rmin = Rmin; sw->dR = dR; sw->dxy = dxy; sw->inc_cos = c;
    sw->Rmax = Rmin + dR * (double)(nr - 1);
    sw->r_dR = 1.0 / dR;
    sw->r_inc = 1.0 / c;
    auto bad = [](double b, double r) {     // Markstein's shortcut needs a normal divisor whose significand is not all ones
        uint64_t bits; memcpy(&bits, &b, 8);
        return ((bits & 0xFFFFFFFFFFFFFull) == 0xFFFFFFFFFFFFFull) || !std::isnormal(b) || !std::isnormal(r);
    };
    sw->true_div = (bad(dR, sw->r_dR) || bad(c, sw->r_inc)) ? 1 : 0;
    (void)p;
    return true;
}

template <typename T>
int do_sample_image(gal_plan* p, const T* image, const SweepParams* sw, int C, double dxy, const T* u, const T* v,
                    const T* re, const T* im, const T* w, int64_t M, double dRA, double dDec, double PA, T* vis,
                    double* chi2_pc, double* chi2_tot, void* stream) {
    if (!prec_ok<T>(p) || (!image && !sw) || !(dxy > 0) || M < 0 || C < 1 || C > p->batch) return GAL_ERR_INVALID_ARGUMENT;
    if (M > 0 && (!u || !v)) return GAL_ERR_INVALID_ARGUMENT;
    const bool chi2 = (vis == nullptr);
    if (chi2 && (!chi2_pc && !chi2_tot)) return GAL_ERR_INVALID_ARGUMENT;
    if (chi2 && M > 0 && (!re || !im || !w)) return GAL_ERR_INVALID_ARGUMENT;
    if (!std::isfinite(dRA) || !std::isfinite(dDec) || !std::isfinite(PA)) return GAL_ERR_INVALID_ARGUMENT;
    // the kernels read the image as complex pairs / 16-byte bulk copies and store visibilities as complex values
    if ((image && !aligned_to(image, 16)) || (vis && !aligned_to(vis, 2 * sizeof(T)))) return GAL_ERR_INVALID_ARGUMENT;
    if (p->viol_host && *(volatile unsigned int*)p->viol_host) {      // an earlier call found the bound uv set changed
        *(volatile unsigned int*)p->viol_host = 0;
        gal_plan_unbind_obs(p);
        return GAL_ERR_BINDING_VIOLATED;
    }
    DeviceGuard g(p->device);
    cudaStream_t st = (cudaStream_t)stream;
    p->last_stream = st;
    return run_call<T>(p, image, sw, C, dxy, u, v, re, im, w, M, dRA, dDec, PA, vis, chi2_pc, chi2_tot, st);
}

// sampleProfile / chi2Profile by the direct Hankel transform (hankel.cuh): one kernel, no transform, nxy unused.
template <typename T>
int do_hankel(gal_plan* p, const T* I, int nr, double Rmin, double dR, const T* u, const T* v, const T* re, const T* im,
              const T* w, int64_t M, double dRA, double dDec, double PA, double inc, T* vis, double* chi2, void* stream) {
    SweepParams sw;
    if (!prec_ok<T>(p) || M < 0 || !sweep_args(p, I, nr, Rmin, dR, 1.0, inc, &sw)) return GAL_ERR_INVALID_ARGUMENT;
    if (!vis && !chi2) return GAL_ERR_INVALID_ARGUMENT;
    if (M > 0 && (!u || !v || (!vis && (!re || !im || !w)))) return GAL_ERR_INVALID_ARGUMENT;
    if (vis && !aligned_to(vis, 2 * sizeof(T))) return GAL_ERR_INVALID_ARGUMENT;
    if (!std::isfinite(dRA) || !std::isfinite(dDec) || !std::isfinite(PA)) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    cudaStream_t st = (cudaStream_t)stream;
    p->last_stream = st;
    if (M == 0) {
        if (chi2) GAL_CUDA(p, cudaMemsetAsync(chi2, 0, sizeof(double), st));
        return GAL_OK;
    }
    int rc;
    if ((rc = reset_call_state(p, st))) return rc;
    p->last_pruned = false; p->last_bound = false; p->last_obs = false; p->last_spec = false; p->spec_mode = 0;
    const CallScalars cs = call_scalars(p, 1.0 / p->nxy, dRA, dDec, PA);      // only the rotation and the phase are used
    return launch_hankel<T>(p, sw, cs, u, v, re, im, w, M, vis, vis ? nullptr : chi2, st);
}

template <typename T>
int do_sweep(gal_plan* p, const T* I, int nr, double Rmin, double dR, double dxy, double inc, T* out, void* stream) {
    SweepParams sw;
    if (!prec_ok<T>(p) || !out || !sweep_args(p, I, nr, Rmin, dR, dxy, inc, &sw)) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    cudaStream_t st = (cudaStream_t)stream;
    p->last_stream = st;
    return launch_sweep<T>(p, sw, out, st);
}

template <typename T>
int do_fft2_shifted(gal_plan* p, const T* image, T* out, void* stream) {
    if (!prec_ok<T>(p) || !image || !out || !aligned_to(image, 16) || !aligned_to(out, 2 * sizeof(T))) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    cudaStream_t st = (cudaStream_t)stream;
    p->last_stream = st;
    p->row_small = false;                                  // whole plane
    int rc = fft2<T>(p, image, nullptr, 1, p->ext_full, st);
    if (rc) return rc;
    return launch_transpose<T>(p, out, st);
}

int grow(gal_plan* p, void** buf, size_t* have, size_t want) {
    if (*have >= want) return GAL_OK;
    if (*buf) { cudaFree(*buf); p->owned_bytes -= *have; *buf = nullptr; *have = 0; }
    GAL_CUDA(p, cudaMalloc(buf, want));
    *have = want;
    p->owned_bytes += want;
    return GAL_OK;
}

// Multi-source composition: one model image, S placements
// (dRA_s, dDec_s, PA_s, scale_s); V = sum_s scale_s V_s by the linearity of the transform.  One FFT, pruned to the
// rotation-invariant extent of the point set (its largest baseline length bounds every placement at once: one
// radius reduction instead of S extent passes; nothing at all on a bound uv set), then ONE sampling launch that
// loops the placements inside the per-point routine and, for chi2, compares the sum with the observations in the
// same kernel.  Lists longer than GAL_MULTI_CHUNK placements go chunk by chunk through vis (chi2: a plan-owned sum).
template <typename T>
int do_multi(gal_plan* p, const T* image, double dxy, const T* u, const T* v, const T* re, const T* im, const T* w,
             int64_t M, int S, const double* dRA, const double* dDec, const double* PA, const double* scale, T* vis,
             double* chi2, void* stream) {
    if (!prec_ok<T>(p) || !image || !(dxy > 0) || M < 0 || S < 1 || S > 4096 || !dRA || !dDec || !PA) return GAL_ERR_INVALID_ARGUMENT;
    if (!vis && !chi2) return GAL_ERR_INVALID_ARGUMENT;
    if (M > 0 && (!u || !v || (chi2 && (!re || !im || !w)))) return GAL_ERR_INVALID_ARGUMENT;
    if (!aligned_to(image, 16) || (vis && !aligned_to(vis, 2 * sizeof(T)))) return GAL_ERR_INVALID_ARGUMENT;
    for (int s = 0; s < S; ++s)
        if (!std::isfinite(dRA[s]) || !std::isfinite(dDec[s]) || !std::isfinite(PA[s]) || (scale && !std::isfinite(scale[s])))
            return GAL_ERR_INVALID_ARGUMENT;
    if (S == 1 && (!scale || scale[0] == 1.0))        // a single placement is the plain call (bit for bit)
        return do_sample_image<T>(p, image, nullptr, 1, dxy, u, v, re, im, w, M, dRA[0], dDec[0], PA[0], vis, chi2, nullptr, stream);
    if (p->viol_host && *(volatile unsigned int*)p->viol_host) {
        *(volatile unsigned int*)p->viol_host = 0;
        gal_plan_unbind_obs(p);
        return GAL_ERR_BINDING_VIOLATED;
    }
    DeviceGuard g(p->device);
    cudaStream_t st = (cudaStream_t)stream;
    p->last_stream = st;
    int rc;
    if (M == 0) {
        if (chi2) GAL_CUDA(p, cudaMemsetAsync(chi2, 0, sizeof(double), st));
        return GAL_OK;
    }
    if ((rc = reset_call_state(p, st))) return rc;
    const CallScalars cs0 = call_scalars(p, dxy, 0.0, 0.0, 0.0);
    p->last_bound = false; p->last_obs = false; p->last_spec = false; p->spec_mode = 0;
    p->last_pruned = want_prune<T>(p, 1, M);
    const int* ext = p->ext_full;
    const bool uv_bound = p->b_u == (const void*)u && p->b_v == (const void*)v && p->b_M == M && p->b_C == 1;
    if (uv_bound && !vis && p->o_buf && p->o_src[2] == (const void*)re && p->o_src[3] == (const void*)im &&
        p->o_src[4] == (const void*)w) {              // bound observation set: the private uv-sorted copy
        const T* o = (const T*)p->o_buf;
        u = o; v = o + M; re = o + 2 * M; im = o + 3 * M; w = o + 4 * M;
        p->last_obs = true;
    }
    if (p->prune_mode != 0 && uv_bound) {
        if ((rc = bound_extent(p, cs0, dxy, st))) return rc;
        p->last_bound = true; p->last_pruned = false;
        ext = p->b_ext_dev;
    } else if (p->last_pruned) {
        if ((rc = launch_extent_radius<T>(p, u, v, M, cs0.ix.du, st))) return rc;
        ext = p->ext;
    }
    p->cur_ext = ext;
    p->row_small = p->last_bound ? p->b_ext[0] < p->nxy / 2 : p->last_pruned;   // (the radius extent is pruned unless the data violate Eq. 19)
    if ((rc = fft2<T>(p, image, nullptr, 1, ext, st))) return rc;
    T* sum = vis;
    if (!vis && S > GAL_MULTI_CHUNK) {                // a long list: the running sum of the chunks
        if ((rc = grow(p, &p->st_vis, &p->st_vis_bytes, (size_t)2 * M * sizeof(T)))) return rc;
        sum = (T*)p->st_vis;
    }
    for (int s0 = 0; s0 < S; s0 += GAL_MULTI_CHUNK) {
        PlacementSet ps;
        ps.S = S - s0 < GAL_MULTI_CHUNK ? S - s0 : GAL_MULTI_CHUNK;
        ps.init_from_vis = s0 > 0;
        for (int s = 0; s < ps.S; ++s) {
            const CallScalars c = call_scalars(p, dxy, dRA[s0 + s], dDec[s0 + s], PA[s0 + s]);
            ps.pl[s] = Placement{c.ix.cos_PA, c.ix.sin_PA, c.dRA_turns, c.dDec_turns, scale ? scale[s0 + s] : 1.0, c.has_phase, 0};
        }
        const bool last = s0 + GAL_MULTI_CHUNK >= S;
        const bool write_vis = vis || !last;
        if ((rc = launch_sample_multi<T>(p, cs0.ix, ps, u, v, re, im, w, M, sum, write_vis, write_vis ? nullptr : chi2, last, st)))
            return rc;
    }
    return GAL_OK;
}

// Host-pointer variant: stage everything through plan-owned device buffers on `stream`.
template <typename T>
int do_host_call(gal_plan* p, const T* image, const T* I, int nr, double Rmin, double dR, double inc, double dxy,
                 const T* u, const T* v, const T* re, const T* im, const T* w, int64_t M, double dRA, double dDec,
                 double PA, T* vis_out, double* chi2_out, void* stream) {
    if (!prec_ok<T>(p) || M < 0 || (!image && !I)) return GAL_ERR_INVALID_ARGUMENT;
    if (!vis_out && !chi2_out) return GAL_ERR_INVALID_ARGUMENT;
    if (M > 0 && (!u || !v || (chi2_out && (!re || !im || !w)))) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n2 = (size_t)p->nxy * p->nxy;
    const size_t img_bytes = image ? n2 * sizeof(T) : (size_t)nr * sizeof(T);
    const int narr = chi2_out ? 5 : 2;
    int rc;
    if ((rc = grow(p, &p->st_image, &p->st_image_bytes, img_bytes))) return rc;
    if ((rc = grow(p, &p->st_pts, &p->st_pts_bytes, (size_t)narr * (size_t)(M > 0 ? M : 1) * sizeof(T)))) return rc;
    if (vis_out && (rc = grow(p, &p->st_out, &p->st_out_bytes, (size_t)2 * (size_t)(M > 0 ? M : 1) * sizeof(T)))) return rc;
    GAL_CUDA(p, cudaMemcpyAsync(p->st_image, image ? (const void*)image : (const void*)I, img_bytes, cudaMemcpyHostToDevice, st));
    T* d = (T*)p->st_pts;
    const T* src[5] = {u, v, re, im, w};
    for (int a = 0; a < narr && M > 0; ++a)
        GAL_CUDA(p, cudaMemcpyAsync(d + (size_t)a * M, src[a], (size_t)M * sizeof(T), cudaMemcpyHostToDevice, st));
    SweepParams sw;
    const SweepParams* swp = nullptr;
    if (!image) {
        if (!sweep_args(p, p->st_image, nr, Rmin, dR, dxy, inc, &sw)) return GAL_ERR_INVALID_ARGUMENT;
        swp = &sw;
    }
    rc = do_sample_image<T>(p, image ? (const T*)p->st_image : nullptr, swp, 1, dxy, d, d + M, d + 2 * M, d + 3 * M,
                            d + 4 * M, M, dRA, dDec, PA, vis_out ? (T*)p->st_out : nullptr,
                            chi2_out ? p->st_chi2 : nullptr, nullptr, stream);
    if (rc) return rc;
    if (vis_out && M > 0)
        GAL_CUDA(p, cudaMemcpyAsync(vis_out, p->st_out, (size_t)2 * M * sizeof(T), cudaMemcpyDeviceToHost, st));
    if (chi2_out) GAL_CUDA(p, cudaMemcpyAsync(chi2_out, p->st_chi2, sizeof(double), cudaMemcpyDeviceToHost, st));
    GAL_CUDA(p, cudaStreamSynchronize(st));
    return GAL_OK;
}

}  // namespace

extern "C" int gal_plan_unbind_uv(gal_plan* p);
extern "C" int gal_plan_unbind_obs(gal_plan* p);

namespace {

template <typename T>
int do_bind_uv(gal_plan* p, const T* u, const T* v, int64_t M, int C, void* stream) {
    if (!prec_ok<T>(p) || !u || !v || M < 1 || C < 1 || C > p->batch) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    cudaStream_t st = (cudaStream_t)stream;
    gal_plan_unbind_obs(p);
    GAL_CUDA(p, cudaMemsetAsync(p->b_r2, 0, 8, st));
    { int rc = launch_uv_radius<T>(p, u, v, (long long)C * M, st); if (rc) return rc; }
    unsigned long long bits = 0;
    GAL_CUDA(p, cudaMemcpyAsync(&bits, p->b_r2, 8, cudaMemcpyDeviceToHost, st));
    GAL_CUDA(p, cudaStreamSynchronize(st));
    double r2; memcpy(&r2, &bits, 8);
    if (!std::isfinite(r2)) return GAL_ERR_INVALID_ARGUMENT;
    p->b_rmax = std::sqrt(r2) * (1.0 + 1e-12);
    p->b_u = u; p->b_v = v; p->b_M = M; p->b_C = C;
    return GAL_OK;
}

template <typename T>
int do_bind_obs(gal_plan* p, const T* u, const T* v, const T* re, const T* im, const T* w, int64_t M, int C, void* stream) {
    if (!re || !im || !w) return GAL_ERR_INVALID_ARGUMENT;
    if (M >= (int64_t)1 << 32) return GAL_ERR_UNSUPPORTED;                  // 32-bit permutation indices
    int rc = do_bind_uv<T>(p, u, v, M, C, stream);                        // validates, leaves r_max and the uv binding
    if (rc) return rc;
    DeviceGuard g(p->device);
    const size_t bytes = (size_t)5 * C * M * sizeof(T);
    if ((rc = grow(p, &p->o_buf, &p->o_bytes, bytes))) { gal_plan_unbind_uv(p); return rc; }
    if ((rc = launch_bind_sort<T>(p, u, v, re, im, w, M, C, p->b_rmax, (T*)p->o_buf, (cudaStream_t)stream))) {
        gal_plan_unbind_obs(p);
        return rc;
    }
    p->o_src[0] = u; p->o_src[1] = v; p->o_src[2] = re; p->o_src[3] = im; p->o_src[4] = w;
    p->o_M = M; p->o_C = C;
    return GAL_OK;
}

}  // namespace

// =============================================================================================
// C ABI
// =============================================================================================
extern "C" {

const char* gal_strerror(int code) {
    switch (code) {
        case GAL_OK: return "ok";
        case GAL_ERR_INVALID_ARGUMENT: return "invalid argument";
        case GAL_ERR_ALLOC: return "allocation failed";
        case GAL_ERR_CUDA: return "CUDA error (see gal_last_cuda_error)";
        case GAL_ERR_UNSUPPORTED: return "unsupported size";
        case GAL_ERR_BINDING_VIOLATED: return "a bound (u, v) set changed after gal_plan_bind_uv / gal_plan_bind_obs";
        case GAL_ERR_TOO_LARGE: return "M exceeds GAL_NOALLOC_MAX_POINTS (1048576): the fixed scratch of the no-allocation entry point cannot hold more partial sums";
        default: return "unknown error";
    }
}

int gal_plan_create(gal_plan** out, int nxy, int batch, int precision_bits, int device) {
    if (!out) return GAL_ERR_INVALID_ARGUMENT;
    *out = nullptr;
    if (!is_pow2(nxy) || nxy < 8 || batch < 1 || (precision_bits != 64 && precision_bits != 32) || device < 0)
        return GAL_ERR_INVALID_ARGUMENT;
    if (nxy > 16384) return GAL_ERR_UNSUPPORTED;
    gal_plan* p = new (std::nothrow) gal_plan();
    if (!p) return GAL_ERR_ALLOC;
    p->nxy = nxy; p->batch = batch; p->bits = precision_bits; p->device = device;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev) { delete p; return GAL_ERR_CUDA; }
    DeviceGuard g(device);
    cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, device);
    p->max_gx = p->sm_count * 8;
    const size_t esz = precision_bits == 64 ? sizeof(double2) : sizeof(float2);
    const size_t work_bytes = (size_t)batch * (nxy / 2 + 1) * nxy * esz;
    const size_t spec_bytes = 2 * work_bytes;
    auto fail = [&](int code, cudaError_t e) { p->last_cuda = (int)e; gal_plan_destroy(p); return code; };
    cudaError_t e;
    if ((e = cudaMalloc(&p->spec, spec_bytes)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc(&p->work, work_bytes)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc(&p->tw, (size_t)nxy * esz)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc((void**)&p->partials, sizeof(double) * (size_t)batch * p->max_gx)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc((void**)&p->tickets, sizeof(unsigned int) * (batch + 1))) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc(&p->call_state, 64)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc(&p->call_init, 32)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc((void**)&p->ext_full, 16)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc((void**)&p->b_ext_dev, 16)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc((void**)&p->b_r2, 8)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMalloc(&p->spec_state, 128)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    if ((e = cudaMemset(p->spec_state, 0, 128)) != cudaSuccess) return fail(GAL_ERR_CUDA, e);
    if ((e = cudaHostAlloc((void**)&p->viol_host, 2 * sizeof(unsigned int), cudaHostAllocMapped)) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    p->viol_host[0] = 0; p->viol_host[1] = 0;          // [1]: extent hint (plan.h row_small)
    if ((e = cudaHostGetDevicePointer((void**)&p->viol_dev, p->viol_host, 0)) != cudaSuccess) return fail(GAL_ERR_CUDA, e);
    p->oob = (unsigned long long*)p->call_state;
    p->ext = (int*)((char*)p->call_state + 8);
    {
        int init[8] = {0, 0, /* ext: */ 1, nxy / 2, nxy / 2 + 1, 0, 0, 0};
        int full[4] = {nxy / 2, 0, nxy - 1, 0};
        if ((e = cudaMemcpy(p->call_init, init, 32, cudaMemcpyHostToDevice)) != cudaSuccess) return fail(GAL_ERR_CUDA, e);
        if ((e = cudaMemcpy(p->call_state, init, 32, cudaMemcpyHostToDevice)) != cudaSuccess) return fail(GAL_ERR_CUDA, e);
        if ((e = cudaMemcpy((char*)p->call_state + 32, init, 32, cudaMemcpyHostToDevice)) != cudaSuccess) return fail(GAL_ERR_CUDA, e);
        if ((e = cudaMemcpy(p->ext_full, full, 16, cudaMemcpyHostToDevice)) != cudaSuccess) return fail(GAL_ERR_CUDA, e);
    }
    if ((e = cudaMalloc((void**)&p->st_chi2, sizeof(double))) != cudaSuccess) return fail(GAL_ERR_ALLOC, e);
    p->owned_bytes = spec_bytes + work_bytes + (size_t)nxy * esz + sizeof(double) * (size_t)batch * p->max_gx +
                     sizeof(unsigned int) * (batch + 1) + 176;
    if ((e = cudaMemset(p->tickets, 0, sizeof(unsigned int) * (batch + 1))) != cudaSuccess) return fail(GAL_ERR_CUDA, e);
    // the workspace starts as zeros (pruned calls leave parts of it unwritten; they are never sampled)
    if ((e = cudaMemset(p->spec, 0, spec_bytes)) != cudaSuccess) return fail(GAL_ERR_CUDA, e);
    // twiddle table exp(-2 pi i m / nxy): evaluated in long double on the host, octant-exact
    std::vector<double> twd((size_t)2 * nxy);
    const long double PI = 3.14159265358979323846264338327950288L;
    for (int m = 0; m < nxy; ++m) {
        long double a = -2.0L * PI * (long double)m / (long double)nxy;
        twd[2 * m] = (double)cosl(a);
        twd[2 * m + 1] = (double)sinl(a);
    }
    if (precision_bits == 64) {
        e = cudaMemcpy(p->tw, twd.data(), sizeof(double) * 2 * nxy, cudaMemcpyHostToDevice);
    } else {
        std::vector<float> twf((size_t)2 * nxy);
        for (size_t i = 0; i < twf.size(); ++i) twf[i] = (float)twd[i];
        e = cudaMemcpy(p->tw, twf.data(), sizeof(float) * 2 * nxy, cudaMemcpyHostToDevice);
    }
    if (e != cudaSuccess) return fail(GAL_ERR_CUDA, e);
    *out = p;
    return GAL_OK;
}

int gal_plan_destroy(gal_plan* p) {
    if (!p) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    cudaFree(p->spec); cudaFree(p->work); cudaFree(p->tw); cudaFree(p->partials); cudaFree(p->tickets);
    for (auto& m : p->tev) cudaEventDestroy(m.ev);
    cudaFree(p->o_buf); if (p->viol_host) cudaFreeHost(p->viol_host);
    cudaFree(p->call_state); cudaFree(p->call_init); cudaFree(p->ext_full); cudaFree(p->b_ext_dev); cudaFree(p->b_r2); cudaFree(p->spec_state); cudaFree(p->st_vis); cudaFree(p->st_image); cudaFree(p->st_pts); cudaFree(p->st_out); cudaFree(p->st_chi2);
    delete p;
    return GAL_OK;
}

int gal_plan_timing_enable(gal_plan* p, int max_calls) {
    if (!p || max_calls < 0 || max_calls > (1 << 20)) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    for (auto& m : p->tev) cudaEventDestroy(m.ev);
    p->tev.clear();
    p->t_calls = 0;
    p->t_on = false;
    p->t_max_calls = max_calls;
    return GAL_OK;
}

int gal_plan_timing_read(gal_plan* p, double* ms_per_kernel, int64_t* calls) {
    if (!p || !ms_per_kernel) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    double acc[4] = {0, 0, 0, 0};
    for (size_t i = 1; i < p->tev.size(); ++i) {
        const gal_plan::Mark &a = p->tev[i - 1], &b = p->tev[i];
        if (a.call != b.call || b.what < 1 || b.what > 4) continue;
        GAL_CUDA(p, cudaEventSynchronize(b.ev));
        float ms = 0;
        GAL_CUDA(p, cudaEventElapsedTime(&ms, a.ev, b.ev));
        acc[b.what - 1] += ms;
    }
    for (int k = 0; k < 4; ++k) ms_per_kernel[k] = p->t_calls ? acc[k] / p->t_calls : 0.0;
    if (calls) *calls = p->t_calls;
    return GAL_OK;
}

int gal_plan_set_pruning(gal_plan* p, int mode) {
    if (!p || mode < 0 || mode > 2) return GAL_ERR_INVALID_ARGUMENT;
    p->prune_mode = mode;
    return GAL_OK;
}

// Tuning options of a plan (the library reads no environment variable).  They select among kernels / launch
// geometries that compute the same thing; no result depends on them beyond the last bits of the transform.
int gal_plan_set_option(gal_plan* p, int option, double value) {
    if (!p || !std::isfinite(value)) return GAL_ERR_INVALID_ARGUMENT;
    const int iv = (int)value;
    switch (option) {
        case GAL_OPT_ROW_MODE: if (iv < -1 || iv > 3) return GAL_ERR_INVALID_ARGUMENT; p->row_mode = iv; break;
        case GAL_OPT_BATCH_CHUNK: if (iv < 0) return GAL_ERR_INVALID_ARGUMENT; p->batch_chunk = iv; break;
        case GAL_OPT_SPECULATE: p->spec_off = (iv == 0); p->spec_valid = false; break;
        case GAL_OPT_SPEC_MIN_BYTES: if (value < 0) return GAL_ERR_INVALID_ARGUMENT; p->spec_min_bytes = value; p->spec_valid = false; break;
        case GAL_OPT_BATCH_CONC: if (iv < 1) return GAL_ERR_INVALID_ARGUMENT; p->batch_conc = iv; break;
        case GAL_OPT_ROW_PREFETCH: if (value < 0) return GAL_ERR_INVALID_ARGUMENT; p->row_pf = value; p->resident.clear(); break;
        case GAL_OPT_ROW_X2_ONE_CTA: p->row_x2_one_cta = (iv != 0); break;
        default: return GAL_ERR_INVALID_ARGUMENT;
    }
    return GAL_OK;
}

int gal_last_uv_extent(gal_plan* p, int* extent) {
    if (!p || !extent) return GAL_ERR_INVALID_ARGUMENT;
    DeviceGuard g(p->device);
    GAL_CUDA(p, cudaStreamSynchronize(p->last_stream));
    if (p->last_bound) { extent[0] = p->b_ext[0]; extent[1] = p->b_ext[1]; extent[2] = p->b_ext[2]; return GAL_OK; }
    if (p->last_spec) { GAL_CUDA(p, cudaMemcpy(extent, p->spec_used(), 3 * sizeof(int), cudaMemcpyDeviceToHost)); return GAL_OK; }
    GAL_CUDA(p, cudaMemcpy(extent, p->last_pruned ? p->ext : p->ext_full, 3 * sizeof(int), cudaMemcpyDeviceToHost));
    return GAL_OK;
}

int gal_get_image_size(const double* u, const double* v, int64_t M, double PB, double f_min, double f_max,
                       int* nxy_out, double* dxy_out) {
    if (!u || !v || M < 1 || !nxy_out || !dxy_out || !std::isfinite(PB)) return GAL_ERR_INVALID_ARGUMENT;
    if (!(f_min > 0)) f_min = 5.0;
    if (!(f_max > 0)) f_max = 2.5;
    double qmin = INFINITY, qmax = 0.0;
    for (int64_t k = 0; k < M; ++k) {
        const double q = std::hypot(u[k], v[k]);
        if (!std::isfinite(q)) return GAL_ERR_INVALID_ARGUMENT;
        qmin = q < qmin ? q : qmin;
        qmax = q > qmax ? q : qmax;
    }
    if (!(qmin > 0)) return GAL_ERR_INVALID_ARGUMENT;
    const double Gamma = 0.6;
    const double duv = PB > 0 ? 1.0 / PB : qmin / (Gamma * f_min);   // Eq. 23 / Eq. 21
    const double n_raw = 2.0 * f_max * qmax / duv;              // Eq. 19
    if (!(n_raw < 1073741824.0)) return GAL_ERR_INVALID_ARGUMENT;
    int n = 2;
    while ((double)n < n_raw) n *= 2;
    *nxy_out = n;
    *dxy_out = 1.0 / ((double)n * duv);                         // Eq. 16
    return GAL_OK;
}

int gal_plan_unbind_uv(gal_plan* p) { return gal_plan_unbind_obs(p); }

int gal_plan_unbind_obs(gal_plan* p) {
    if (!p) return GAL_ERR_INVALID_ARGUMENT;
    p->b_u = p->b_v = nullptr; p->b_M = 0; p->b_C = 0; p->b_dxy = 0.0; p->last_bound = false;
    for (auto& q : p->o_src) q = nullptr;
    p->o_M = 0; p->o_C = 0; p->last_obs = false;         // (the private copy's memory is kept for the next binding)
    if (p->viol_host) *(volatile unsigned int*)p->viol_host = 0;
    return GAL_OK;
}

int64_t gal_last_extent_violations(gal_plan* p) {
    if (!p) return -1;
    if (!p->last_bound) return 0;
    DeviceGuard g(p->device);
    unsigned long long h = 0;
    if (cudaStreamSynchronize(p->last_stream) != cudaSuccess) return -1;
    if (cudaMemcpy(&h, (char*)p->oob + 24, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return (int64_t)h;
}

size_t gal_plan_workspace_bytes(const gal_plan* p) { return p ? p->owned_bytes : 0; }
int gal_last_cuda_error(const gal_plan* p) { return p ? p->last_cuda : 0; }
int64_t gal_plan_launch_count(const gal_plan* p) { return p ? p->launches : -1; }

int64_t gal_last_oob_count(gal_plan* p) {
    if (!p) return -1;
    DeviceGuard g(p->device);
    unsigned long long h = 0;
    if (cudaStreamSynchronize(p->last_stream) != cudaSuccess) return -1;
    if (cudaMemcpy(&h, p->oob, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return (int64_t)h;
}

#define GAL_DEFINE_PRECISION(SFX, T)                                                                                  \
    int gal_plan_bind_uv_##SFX(gal_plan* p, const T* u, const T* v, int64_t M, int C, void* stream) {                 \
        return do_bind_uv<T>(p, u, v, M, C, stream);                                                                  \
    }                                                                                                                 \
    int gal_plan_bind_obs_##SFX(gal_plan* p, const T* u, const T* v, const T* re, const T* im, const T* w, int64_t M, \
                                int C, void* stream) {                                                                \
        return do_bind_obs<T>(p, u, v, re, im, w, M, C, stream);                                                      \
    }                                                                                                                 \
    int gal_sweep_##SFX(gal_plan* p, const T* I, int nr, double Rmin, double dR, double dxy, double inc, T* out,      \
                        void* stream) {                                                                               \
        return do_sweep<T>(p, I, nr, Rmin, dR, dxy, inc, out, stream);                                                \
    }                                                                                                                 \
    int gal_fft2_shifted_##SFX(gal_plan* p, const T* image, T* out, void* stream) {                                   \
        return do_fft2_shifted<T>(p, image, out, stream);                                                             \
    }                                                                                                                 \
    int gal_sample_image_##SFX(gal_plan* p, const T* image, double dxy, const T* u, const T* v, int64_t M,            \
                               double dRA, double dDec, double PA, T* vis, void* stream) {                            \
        if (!image || (M > 0 && !vis)) return GAL_ERR_INVALID_ARGUMENT;                                               \
        if (M == 0) return GAL_OK;                                                                                    \
        return do_sample_image<T>(p, image, nullptr, 1, dxy, u, v, nullptr, nullptr, nullptr, M, dRA, dDec, PA, vis,  \
                                  nullptr, nullptr, stream);                                                          \
    }                                                                                                                 \
    int gal_chi2_image_##SFX(gal_plan* p, const T* image, double dxy, const T* u, const T* v, const T* re,            \
                             const T* im, const T* w, int64_t M, double dRA, double dDec, double PA, double* chi2,    \
                             void* stream) {                                                                          \
        if (!image || !chi2) return GAL_ERR_INVALID_ARGUMENT;                                                         \
        return do_sample_image<T>(p, image, nullptr, 1, dxy, u, v, re, im, w, M, dRA, dDec, PA, nullptr, chi2,        \
                                  nullptr, stream);                                                                   \
    }                                                                                                                 \
    int gal_sample_profile_##SFX(gal_plan* p, const T* I, int nr, double Rmin, double dR, double dxy, const T* u,     \
                                 const T* v, int64_t M, double dRA, double dDec, double PA, double inc, T* vis,       \
                                 void* stream) {                                                                      \
        SweepParams sw;                                                                                               \
        if (!sweep_args(p, I, nr, Rmin, dR, dxy, inc, &sw) || (M > 0 && !vis)) return GAL_ERR_INVALID_ARGUMENT;       \
        if (M == 0) return GAL_OK;                                                                                    \
        return do_sample_image<T>(p, nullptr, &sw, 1, dxy, u, v, nullptr, nullptr, nullptr, M, dRA, dDec, PA, vis,    \
                                  nullptr, nullptr, stream);                                                          \
    }                                                                                                                 \
    int gal_chi2_profile_##SFX(gal_plan* p, const T* I, int nr, double Rmin, double dR, double dxy, const T* u,       \
                               const T* v, const T* re, const T* im, const T* w, int64_t M, double dRA, double dDec,  \
                               double PA, double inc, double* chi2, void* stream) {                                   \
        SweepParams sw;                                                                                               \
        if (!sweep_args(p, I, nr, Rmin, dR, dxy, inc, &sw) || !chi2) return GAL_ERR_INVALID_ARGUMENT;                 \
        return do_sample_image<T>(p, nullptr, &sw, 1, dxy, u, v, re, im, w, M, dRA, dDec, PA, nullptr, chi2, nullptr, \
                                  stream);                                                                            \
    }                                                                                                                 \
    int gal_sample_profile_hankel_##SFX(gal_plan* p, const T* I, int nr, double Rmin, double dR, const T* u, const T* v,  \
                                        int64_t M, double dRA, double dDec, double PA, double inc, T* vis, void* stream) { \
        if (M > 0 && !vis) return GAL_ERR_INVALID_ARGUMENT;                                                           \
        if (M == 0) return GAL_OK;                                                                                    \
        return do_hankel<T>(p, I, nr, Rmin, dR, u, v, nullptr, nullptr, nullptr, M, dRA, dDec, PA, inc, vis, nullptr,  \
                            stream);                                                                                  \
    }                                                                                                                 \
    int gal_chi2_profile_hankel_##SFX(gal_plan* p, const T* I, int nr, double Rmin, double dR, const T* u, const T* v, \
                                      const T* re, const T* im, const T* w, int64_t M, double dRA, double dDec,       \
                                      double PA, double inc, double* chi2, void* stream) {                            \
        if (!chi2) return GAL_ERR_INVALID_ARGUMENT;                                                                   \
        return do_hankel<T>(p, I, nr, Rmin, dR, u, v, re, im, w, M, dRA, dDec, PA, inc, nullptr, chi2, stream);       \
    }                                                                                                                 \
    int gal_chi2_image_batch_##SFX(gal_plan* p, const T* images, int C, double dxy, const T* u, const T* v,           \
                                   const T* re, const T* im, const T* w, int64_t M, double dRA, double dDec,          \
                                   double PA, double* chi2_pc, double* chi2_tot, void* stream) {                      \
        if (!p || !images || !chi2_pc || C < 1) return GAL_ERR_INVALID_ARGUMENT;                                      \
        return do_sample_image<T>(p, images, nullptr, C, dxy, u, v, re, im, w, M, dRA, dDec, PA, nullptr, chi2_pc,    \
                                  chi2_tot, stream);                                                                  \
    }                                                                                                                 \
    int gal_chi2_image_sets_##SFX(gal_plan* p, const T* image, int K, double dxy, const T* u, const T* v,             \
                                  const T* re, const T* im, const T* w, int64_t M, double dRA, double dDec,           \
                                  double PA, double* chi2_ps, double* chi2_tot, void* stream) {                       \
        if (!p || !image || !chi2_ps || K < 1) return GAL_ERR_INVALID_ARGUMENT;                                       \
        p->shared_spec = true;                                                                                        \
        const int rc = do_sample_image<T>(p, image, nullptr, K, dxy, u, v, re, im, w, M, dRA, dDec, PA, nullptr,      \
                                          chi2_ps, chi2_tot, stream);                                                 \
        p->shared_spec = false;                                                                                       \
        return rc;                                                                                                    \
    }                                                                                                                 \
    int gal_sample_image_multi_##SFX(gal_plan* p, const T* image, double dxy, const T* u, const T* v, int64_t M,      \
                                     int S, const double* dRA, const double* dDec, const double* PA,                  \
                                     const double* scale, T* vis, void* stream) {                                     \
        if (M > 0 && !vis) return GAL_ERR_INVALID_ARGUMENT;                                                           \
        if (M == 0) return GAL_OK;                                                                                    \
        return do_multi<T>(p, image, dxy, u, v, nullptr, nullptr, nullptr, M, S, dRA, dDec, PA, scale, vis, nullptr,  \
                           stream);                                                                                   \
    }                                                                                                                 \
    int gal_chi2_image_multi_##SFX(gal_plan* p, const T* image, double dxy, const T* u, const T* v, const T* re,      \
                                   const T* im, const T* w, int64_t M, int S, const double* dRA, const double* dDec,  \
                                   const double* PA, const double* scale, double* chi2, void* stream) {               \
        if (!chi2) return GAL_ERR_INVALID_ARGUMENT;                                                                   \
        return do_multi<T>(p, image, dxy, u, v, re, im, w, M, S, dRA, dDec, PA, scale, nullptr, chi2, stream);        \
    }                                                                                                                 \
    int gal_chi2_image_host_##SFX(gal_plan* p, const T* image, double dxy, const T* u, const T* v, const T* re,       \
                                  const T* im, const T* w, int64_t M, double dRA, double dDec, double PA,             \
                                  double* chi2, void* stream) {                                                       \
        if (!image || !chi2) return GAL_ERR_INVALID_ARGUMENT;                                                         \
        return do_host_call<T>(p, image, nullptr, 0, 0, 0, 0, dxy, u, v, re, im, w, M, dRA, dDec, PA, nullptr, chi2,  \
                               stream);                                                                               \
    }                                                                                                                 \
    int gal_sample_image_host_##SFX(gal_plan* p, const T* image, double dxy, const T* u, const T* v, int64_t M,       \
                                    double dRA, double dDec, double PA, T* vis, void* stream) {                       \
        if (!image || !vis) return GAL_ERR_INVALID_ARGUMENT;                                                          \
        return do_host_call<T>(p, image, nullptr, 0, 0, 0, 0, dxy, u, v, nullptr, nullptr, nullptr, M, dRA, dDec, PA, \
                               vis, nullptr, stream);                                                                 \
    }                                                                                                                 \
    int gal_chi2_profile_host_##SFX(gal_plan* p, const T* I, int nr, double Rmin, double dR, double dxy, const T* u,  \
                                    const T* v, const T* re, const T* im, const T* w, int64_t M, double dRA,          \
                                    double dDec, double PA, double inc, double* chi2, void* stream) {                 \
        if (!I || !chi2 || nr < 2) return GAL_ERR_INVALID_ARGUMENT;                                                   \
        return do_host_call<T>(p, nullptr, I, nr, Rmin, dR, inc, dxy, u, v, re, im, w, M, dRA, dDec, PA, nullptr,     \
                               chi2, stream);                                                                         \
    }                                                                                                                 \
    int gal_sample_profile_host_##SFX(gal_plan* p, const T* I, int nr, double Rmin, double dR, double dxy,            \
                                      const T* u, const T* v, int64_t M, double dRA, double dDec, double PA,          \
                                      double inc, T* vis, void* stream) {                                             \
        if (!I || !vis || nr < 2) return GAL_ERR_INVALID_ARGUMENT;                                                    \
        return do_host_call<T>(p, nullptr, I, nr, Rmin, dR, inc, dxy, u, v, nullptr, nullptr, nullptr, M, dRA, dDec,  \
                               PA, vis, nullptr, stream);                                                             \
    }

GAL_DEFINE_PRECISION(f64, double)
GAL_DEFINE_PRECISION(f32, float)

}  // extern "C"
