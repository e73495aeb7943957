// C ABI of libglad (include/glad.h): context, static data, argument checks, scratch, launch order.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "glad_internal.h"

static glad_status fail(glad_ctx* c, glad_status st, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return st;
}
static glad_status cuda_fail(glad_ctx* c, cudaError_t e, const char* what) {
    return fail(c, GLAD_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}
#define CU(call, what)                                           \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return cuda_fail(c, e__, what);  \
    } while (0)

// Grow-only scratch.  A growth synchronises both streams (the old block may be in use) -- the one hidden host sync of a batch
// call, on its first use or when a larger batch arrives.  `exact`: no 25 % headroom (blocks sized against a caller's limit).
template <typename T>
static glad_status grow(glad_ctx* c, T** p, size_t* cap, size_t need, bool exact = false) {
    if (need <= *cap) return GLAD_OK;
    // the stream may still be using the old block: free is stream-ordered w.r.t. nothing, so sync first
    cudaStreamSynchronize(c->stream);
    if (c->side_stream) cudaStreamSynchronize(c->side_stream);
    if (*p) cudaFree(*p);
    *p = nullptr;
    *cap = 0;
    size_t n = exact ? need : need + need / 4;
    if (cudaMalloc((void**)p, n * sizeof(T)) != cudaSuccess) {
        cudaGetLastError();
        return fail(c, GLAD_ENOMEM, "cudaMalloc of %zu bytes failed", n * sizeof(T));
    }
    *cap = n;
    return GLAD_OK;
}

extern "C" {

const char* glad_version(void) { return "libglad 0.1 (sm_100a)"; }

glad_status glad_create(glad_ctx** out, int device, void* cuda_stream) {
    if (!out) return GLAD_EINVAL;
    *out = nullptr;
    glad_ctx* c = new glad_ctx();
    memset(c, 0, sizeof(*c));
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    int major = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e != cudaSuccess || major != 10) {
        cudaGetLastError();
        delete c;
        return GLAD_ECUDA;
    }
    DeviceScope ds(c);
    c->jam_simt = 0; c->jam_terms = 2; c->jam_flush = 0; c->jam_slices = 0;
    c->lens_stream = c->stream;
    if (cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        c->side_ok = 0;
    } else {
        c->side_ok = 1;
    }
    c->overlap = c->side_ok;
    if (lens_noalloc_setup(c) != cudaSuccess) cudaGetLastError();     // glad_lens_image_noalloc then reports GLAD_ESTATE
    *out = c;
    return GLAD_OK;
}

static void free_kin(glad_ctx* c) {
    void* ps[] = {c->d_xf2, c->d_yf2, c->d_xf, c->d_yf, c->d_foldx, c->d_foldy, c->d_unfoldx, c->d_unfoldy,
                  c->d_binw, c->d_bin_cnt, c->d_binw_ptr, c->d_binw_nz};
    for (void* p : ps) if (p) cudaFree(p);
    c->d_xf2 = c->d_yf2 = c->d_xf = c->d_yf = nullptr;
    c->d_foldx = c->d_foldy = c->d_unfoldx = c->d_unfoldy = nullptr;
    c->d_binw = nullptr;
    c->d_bin_cnt = nullptr;
    c->d_binw_ptr = nullptr;
    c->d_binw_nz = nullptr;
}

void glad_destroy(glad_ctx* c) {
    if (!c) return;
    {
    DeviceScope ds(c);
    cudaStreamSynchronize(c->stream);
    if (c->side_stream) { cudaStreamSynchronize(c->side_stream); cudaStreamDestroy(c->side_stream); }
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    free_kin(c);
    void* ps[] = {c->d_psf, c->d_lens_const, c->d_jam_tab, c->d_partial, c->d_tmp, c->d_tmpflags, c->d_stage, c->d_model, c->d_qtmp, c->d_pix,
                  c->d_sph_tab, c->d_sph_rat, c->d_cse64, c->d_cse32};
    for (void* p : ps) if (p) cudaFree(p);
    for (cudaEvent_t e : c->prof_ev) if (e) cudaEventDestroy(e);
    }
    delete c;
}

glad_status glad_profile_enable(glad_ctx* c, int on) {
    if (!c) return GLAD_EINVAL;
    c->prof_on = on != 0;
    return GLAD_OK;
}

glad_status glad_profile_read(glad_ctx* c, double* ms_out, long* count_out) {
    if (!c || !ms_out || !count_out) return GLAD_EINVAL;
    DeviceScope ds(c);
    CU(cudaStreamSynchronize(c->stream), "profile sync");
    for (int i = 0; i < c->prof_n; ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]) == cudaSuccess) {
            c->prof_ms[c->prof_id[i]] += ms;
            c->prof_cnt[c->prof_id[i]] += 1;
        }
    }
    c->prof_n = 0;
    for (int k = 0; k < GLAD_NKERNELS; ++k) {
        ms_out[k] = c->prof_ms[k]; count_out[k] = c->prof_cnt[k];
        c->prof_ms[k] = 0.0; c->prof_cnt[k] = 0;
    }
    return GLAD_OK;
}

glad_status glad_set_light_profiles(glad_ctx* c, int source_kind, int lens1_kind, int lens2_kind) {
    if (!c) return GLAD_EINVAL;
    const int k[3] = {source_kind, lens1_kind, lens2_kind};
    int bits = 0;
    for (int i = 0; i < 3; ++i) {
        if (k[i] != GLAD_LIGHT_SERSIC && k[i] != GLAD_LIGHT_CHAMELEON) return fail(c, GLAD_EINVAL, "glad_set_light_profiles: kind %d", k[i]);
        if (k[i] == GLAD_LIGHT_CHAMELEON) bits |= 1 << i;
    }
    c->light_kinds = bits;
    return GLAD_OK;
}

glad_status glad_set_mass_sheet(glad_ctx* c, const float* d_lambda, int n_lambda, float r_core, float r_tr, int n_sheet, float sigma_lo, float sigma_hi) {
    if (!c) return GLAD_EINVAL;
    if (!d_lambda) { c->d_lambda = nullptr; return GLAD_OK; }
    if (n_lambda <= 0) return fail(c, GLAD_EINVAL, "glad_set_mass_sheet: n_lambda = %d", n_lambda);
    if (!(r_core > 0.f) || !(r_tr > r_core)) return fail(c, GLAD_EINVAL, "glad_set_mass_sheet: radii %g, %g", r_core, r_tr);
    if (n_sheet < 2 || !(sigma_lo > 0.f) || !(sigma_hi > sigma_lo)) return fail(c, GLAD_EINVAL, "glad_set_mass_sheet: %d Gaussians on [%g, %g]", n_sheet, sigma_lo, sigma_hi);
    if (n_sheet > GLAD_MAX_GAUSS) return fail(c, GLAD_ESHAPE, "glad_set_mass_sheet: more than GLAD_MAX_GAUSS Gaussians");
    c->d_lambda = d_lambda;
    c->n_lambda = n_lambda;
    c->ms_rc = r_core; c->ms_rt = r_tr; c->ms_n = n_sheet; c->ms_lo = sigma_lo; c->ms_hi = sigma_hi;
    return GLAD_OK;
}

glad_status glad_set_jam_options(glad_ctx* c, int path, int bf16_terms, int flush_chunks, int k_slices) {
    if (!c) return GLAD_EINVAL;
    if (path != GLAD_JAM_AUTO && path != GLAD_JAM_SIMT) return fail(c, GLAD_EINVAL, "glad_set_jam_options: path %d", path);
    if (bf16_terms != 0 && bf16_terms != 2 && bf16_terms != 3) return fail(c, GLAD_EINVAL, "glad_set_jam_options: %d bf16 terms (2 or 3)", bf16_terms);
    if (flush_chunks < 0 || k_slices < 0) return fail(c, GLAD_EINVAL, "glad_set_jam_options: negative option");
    c->jam_simt = path == GLAD_JAM_SIMT;
    c->jam_terms = bf16_terms ? bf16_terms : 2;
    c->jam_flush = flush_chunks;
    c->jam_slices = k_slices;
    return GLAD_OK;
}

glad_status glad_set_enfw(glad_ctx* c, const float* d_enfw, int n_enfw, int n_cse, const double* h_A, const double* h_s, int n_gauss,
                          float sigma_lo, float sigma_hi) {
    if (!c) return GLAD_EINVAL;
    if (!d_enfw) { c->d_enfw = nullptr; return GLAD_OK; }
    if (n_enfw <= 0 || !h_A || !h_s) return fail(c, GLAD_EINVAL, "glad_set_enfw: n = %d / null table", n_enfw);
    if (n_cse < 1 || n_cse > GLAD_MAX_CSE) return fail(c, GLAD_ESHAPE, "glad_set_enfw: %d core-steep ellipsoids (1..GLAD_MAX_CSE)", n_cse);
    if (n_gauss < 2 || !(sigma_lo > 0.f) || !(sigma_hi > sigma_lo)) return fail(c, GLAD_EINVAL, "glad_set_enfw: %d Gaussians on [%g, %g]", n_gauss, sigma_lo, sigma_hi);
    if (n_gauss > GLAD_MAX_GAUSS) return fail(c, GLAD_ESHAPE, "glad_set_enfw: more than GLAD_MAX_GAUSS Gaussians");
    double2 t64[GLAD_MAX_CSE];
    float2 t32[GLAD_MAX_CSE];
    for (int i = 0; i < n_cse; ++i) {
        if (!(h_s[i] > 0.0) || !isfinite(h_A[i])) return fail(c, GLAD_EINVAL, "glad_set_enfw: table entry %d = (%g, %g)", i, h_A[i], h_s[i]);
        t64[i] = make_double2(h_A[i], h_s[i]);
        t32[i] = make_float2((float)(h_A[i] / h_s[i]), (float)h_s[i]);
    }
    DeviceScope ds(c);
    CU(cudaStreamSynchronize(c->stream), "sync");
    if (c->side_stream) CU(cudaStreamSynchronize(c->side_stream), "sync");
    if (!c->d_cse64) CU(cudaMalloc((void**)&c->d_cse64, sizeof(double2) * GLAD_MAX_CSE), "cudaMalloc CSE table");
    if (!c->d_cse32) CU(cudaMalloc((void**)&c->d_cse32, sizeof(float2) * GLAD_MAX_CSE), "cudaMalloc CSE table");
    CU(cudaMemcpy(c->d_cse64, t64, sizeof(double2) * n_cse, cudaMemcpyHostToDevice), "copy CSE table");
    CU(cudaMemcpy(c->d_cse32, t32, sizeof(float2) * n_cse, cudaMemcpyHostToDevice), "copy CSE table");
    c->d_enfw = d_enfw; c->n_enfw = n_enfw; c->ncse = n_cse;
    c->nf_n = n_gauss; c->nf_lo = sigma_lo; c->nf_hi = sigma_hi;
    return GLAD_OK;
}

glad_status glad_set_overlap(glad_ctx* c, int on) {
    if (!c) return GLAD_EINVAL;
    if (on && !c->side_ok) return fail(c, GLAD_ESTATE, "glad_set_overlap: no side stream");
    c->overlap = on ? 1 : 0;
    return GLAD_OK;
}

const char* glad_last_error(const glad_ctx* c) { return c ? c->err : "null context"; }
long glad_launch_count(const glad_ctx* c) { return c ? c->launches : 0; }

double glad_bh_theta2(double mbh_msun, double ddt_mpc, double z_d) {
    const double G = 0.004301, ckms = 299792.458, PI = 3.14159265358979323846;
    double rad2 = 4.0 * G * mbh_msun * (1.0 + z_d) / (ckms * ckms * ddt_mpc * 1e6);
    double as = 648000.0 / PI;
    return rad2 * as * as;
}

glad_status glad_set_image_data(glad_ctx* c, const glad_image_grid* g, const float* d_data, const float* d_ivar,
                                const float* d_psf, int kpsf) {
    if (!c) return GLAD_EINVAL;
    if (!g || !d_psf) return fail(c, GLAD_EINVAL, "glad_set_image_data: null grid or psf");
    if (g->nx <= 0 || g->ny <= 0 || g->supersample <= 0 || !(g->pix > 0.f))
        return fail(c, GLAD_EINVAL, "glad_set_image_data: bad grid %dx%d s=%d pix=%g", g->nx, g->ny, g->supersample, g->pix);
    if ((long)g->nx * g->ny > GLAD_MAX_IMAGE_PIXELS)
        return fail(c, GLAD_ESHAPE, "glad_set_image_data: %dx%d pixels exceed GLAD_MAX_IMAGE_PIXELS", g->nx, g->ny);
    if (kpsf <= 0 || (kpsf % 2) == 0) return fail(c, GLAD_EINVAL, "glad_set_image_data: kpsf must be odd, got %d", kpsf);
    if (kpsf > GLAD_MAX_PSF) return fail(c, GLAD_ESHAPE, "glad_set_image_data: kpsf %d > GLAD_MAX_PSF", kpsf);
    if ((d_data == nullptr) != (d_ivar == nullptr)) return fail(c, GLAD_EINVAL, "glad_set_image_data: data and ivar go together");
    {
        const size_t need = lens_image_smem_bytes(g->nx, g->ny, kpsf);
        if (need > (size_t)glad_smem_dynamic_max(c))
            return fail(c, GLAD_ESHAPE, "glad_set_image_data: a %d x %d image with a %d x %d PSF needs %zu bytes of shared memory (rows padded by the PSF halo), limit %d",
                        g->nx, g->ny, kpsf, kpsf, need, glad_smem_dynamic_max(c));
    }
    DeviceScope ds(c);
    if (!c->d_psf) CU(cudaMalloc((void**)&c->d_psf, sizeof(float) * GLAD_MAX_PSF * GLAD_MAX_PSF), "cudaMalloc psf");
    CU(cudaMemcpyAsync(c->d_psf, d_psf, sizeof(float) * kpsf * kpsf, cudaMemcpyDeviceToDevice, c->stream), "copy psf");
    c->grid = *g;
    c->d_data = d_data;
    c->d_ivar = d_ivar;
    c->kpsf = kpsf;
    c->have_image = true;
    return GLAD_OK;
}

}  // extern "C"

// fold one axis: returns folded length; fills fold[n] (full -> folded), coords of the folded axis, unfold[2*nf]
static int fold_axis(const std::vector<float>& x, std::vector<int>& fold, std::vector<float>& xf, std::vector<int>& unfold) {
    int n = (int)x.size();
    bool sym = n > 1;
    for (int i = 0; i < n && sym; ++i) sym = (x[i] == -x[n - 1 - i]);
    fold.assign(n, 0);
    if (!sym) {
        xf = x;
        unfold.assign(2 * n, -1);
        for (int i = 0; i < n; ++i) { fold[i] = i; unfold[2 * i] = i; }
        return n;
    }
    int nf = (n + 1) / 2, h = n / 2;   // folded index 0 = innermost
    xf.assign(nf, 0.f);
    unfold.assign(2 * nf, -1);
    for (int i = 0; i < n; ++i) {
        int f = (i >= h) ? i - h : (n - 1 - i) - h;   // n odd: centre i = h -> 0
        fold[i] = f;
        xf[f] = fabsf(x[i]);
        if (unfold[2 * f] < 0) unfold[2 * f] = i; else unfold[2 * f + 1] = i;
    }
    return nf;
}

template <typename T>
static cudaError_t upload(T** dst, const std::vector<T>& v) {
    cudaError_t e = cudaMalloc((void**)dst, sizeof(T) * (v.size() ? v.size() : 1));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dst, v.data(), sizeof(T) * v.size(), cudaMemcpyHostToDevice);
}

extern "C" {

glad_status glad_set_kin_data(glad_ctx* c, const glad_sky_grid* g, const int32_t* d_bin_id, int nbins, const float* d_kernel,
                              int kk, const float* d_vobs, const float* d_vivar, const float* d_un, const float* d_uw, int nu) {
    if (!c) return GLAD_EINVAL;
    if (!g || !g->d_xs || !g->d_ys || !d_bin_id || !d_kernel || !d_un || !d_uw)
        return fail(c, GLAD_EINVAL, "glad_set_kin_data: null pointer");
    if (g->nx <= 0 || g->ny <= 0 || nbins <= 0 || nu <= 0) return fail(c, GLAD_EINVAL, "glad_set_kin_data: bad sizes");
    if (g->nx > GLAD_MAX_SKY || g->ny > GLAD_MAX_SKY || nbins > GLAD_MAX_BINS || nu > GLAD_MAX_NODES)
        return fail(c, GLAD_ESHAPE, "glad_set_kin_data: grid %dx%d / nbins %d / nu %d exceed the limits", g->nx, g->ny, nbins, nu);
    if (kk <= 0 || (kk % 2) == 0) return fail(c, GLAD_EINVAL, "glad_set_kin_data: kk must be odd, got %d", kk);
    if (kk > GLAD_MAX_PSF) return fail(c, GLAD_ESHAPE, "glad_set_kin_data: kk %d > GLAD_MAX_PSF", kk);
    if ((d_vobs == nullptr) != (d_vivar == nullptr)) return fail(c, GLAD_EINVAL, "glad_set_kin_data: vrms_obs and vrms_ivar go together");
    DeviceScope ds(c);
    CU(cudaStreamSynchronize(c->stream), "sync");
    std::vector<float> xs(g->nx), ys(g->ny);
    std::vector<int32_t> bins((size_t)g->nx * g->ny);
    CU(cudaMemcpy(xs.data(), g->d_xs, sizeof(float) * g->nx, cudaMemcpyDeviceToHost), "copy xs");
    CU(cudaMemcpy(ys.data(), g->d_ys, sizeof(float) * g->ny, cudaMemcpyDeviceToHost), "copy ys");
    CU(cudaMemcpy(bins.data(), d_bin_id, sizeof(int32_t) * bins.size(), cudaMemcpyDeviceToHost), "copy bin_id");
    std::vector<int> cnt(nbins, 0);
    for (int32_t l : bins) {
        if (l >= nbins) return fail(c, GLAD_EINVAL, "glad_set_kin_data: bin id %d >= nbins %d", (int)l, nbins);
        if (l >= 0) cnt[l]++;
    }
    std::vector<int> fx, fy, ux, uy;
    std::vector<float> xf, yf;
    int nxf = fold_axis(xs, fx, xf, ux), nyf = fold_axis(ys, fy, yf, uy);
    int tiles = ((nxf + JQ_T - 1) / JQ_T) * ((nyf + JQ_T - 1) / JQ_T);
    if (tiles > 512) return fail(c, GLAD_ESHAPE, "glad_set_kin_data: folded grid %dx%d needs %d thread tiles (> 512)", nxf, nyf, tiles);
    {
        // jam_post_kernel stages both folded maps plus (nxf + nyf) floats per luminous Gaussian: necessary condition here
        // (one Gaussian), the exact one in the batch call, which knows n_lum
        const size_t need = jam_post_smem_bytes(nxf, nyf, 1);
        if (need > (size_t)glad_smem_dynamic_max(c))
            return fail(c, GLAD_ESHAPE, "glad_set_kin_data: folded grid %dx%d needs %zu bytes of shared memory in the binning kernel, limit %d",
                        nxf, nyf, need, glad_smem_dynamic_max(c));
    }
    std::vector<float> xf2(nxf), yf2(nyf);
    for (int i = 0; i < nxf; ++i) xf2[i] = xf[i] * xf[i];
    for (int i = 0; i < nyf; ++i) yf2[i] = yf[i] * yf[i];
    free_kin(c);
    c->have_kin = false;
    CU(upload(&c->d_xf, xf), "upload"); CU(upload(&c->d_yf, yf), "upload");
    CU(upload(&c->d_xf2, xf2), "upload"); CU(upload(&c->d_yf2, yf2), "upload");
    CU(upload(&c->d_foldx, fx), "upload"); CU(upload(&c->d_foldy, fy), "upload");
    CU(upload(&c->d_unfoldx, ux), "upload"); CU(upload(&c->d_unfoldy, uy), "upload");
    CU(upload(&c->d_bin_cnt, cnt), "upload");
    CU(cudaMalloc((void**)&c->d_binw, sizeof(float) * (size_t)nbins * nxf * nyf), "cudaMalloc bin weights");
    c->nx = g->nx; c->ny = g->ny; c->nxf = nxf; c->nyf = nyf; c->nbins = nbins; c->kk = kk; c->nu = nu;
    c->d_xs = g->d_xs; c->d_ys = g->d_ys; c->d_bin_id = d_bin_id; c->d_kernel = d_kernel;
    c->d_vobs = d_vobs; c->d_vivar = d_vivar; c->d_un = d_un; c->d_uw = d_uw;
    CU(launch_kin_weights(c), "kin_weights_kernel");
    CU(cudaStreamSynchronize(c->stream), "kin_weights_kernel");
    {
        // compact the static weights: jam_post_kernel walks only the non-zero entries of each bin's row
        const size_t npf = (size_t)nxf * nyf;
        std::vector<float> W((size_t)nbins * npf);
        CU(cudaMemcpy(W.data(), c->d_binw, sizeof(float) * W.size(), cudaMemcpyDeviceToHost), "copy bin weights");
        std::vector<int> ptr(nbins + 1, 0);
        std::vector<float2> nz;
        for (int l = 0; l < nbins; ++l) {
            for (size_t i = 0; i < npf; ++i) {
                const float w = W[(size_t)l * npf + i];
                if (w != 0.f) { float2 e; int idx = (int)i; memcpy(&e.x, &idx, sizeof(int)); e.y = w; nz.push_back(e); }
            }
            ptr[l + 1] = (int)nz.size();
        }
        CU(upload(&c->d_binw_ptr, ptr), "upload");
        CU(upload(&c->d_binw_nz, nz), "upload");
    }
    c->have_kin = true;
    return GLAD_OK;
}

}  // extern "C"

static glad_status lens_impl(glad_ctx* c, const float* d_lens, int B, float* d_images, float* d_chi2, int32_t* d_flags) {
    if (!c->have_image) return fail(c, GLAD_ESTATE, "lens: glad_set_image_data not called");
    if (c->d_lambda && B > c->n_lambda) return fail(c, GLAD_EINVAL, "lens: batch of %d vectors but the mass sheet has %d lambdas", B, c->n_lambda);
    if (c->d_enfw && B > c->n_enfw) return fail(c, GLAD_EINVAL, "lens: batch of %d vectors but %d eNFW halos", B, c->n_enfw);
    if (d_chi2 && !c->d_data) return fail(c, GLAD_ESTATE, "lens: chi2 requested but no data/ivar set");
    glad_status st = grow(c, &c->d_lens_const, &c->lens_const_cap, (size_t)B * LC_SIZE);
    if (st != GLAD_OK) return st;
    CU(launch_lens_prep(c, d_lens, B), "lens_prep_kernel");
    CU(launch_lens_image(c, B, d_images, d_chi2, d_flags), "lens_image_kernel");
    return GLAD_OK;
}

static glad_status jam_impl(glad_ctx* c, const float* d_dyn, int B, const float* d_lum, int nl, long lum_stride,
                            const float* d_mass, int nm, long mass_stride, const float* d_beta, int per_gaussian,
                            float* d_vrms, float* d_chi2, float* d_v2map, int32_t* d_flags) {
    if (!c->have_kin) return fail(c, GLAD_ESTATE, "jam: glad_set_kin_data not called");
    if (d_chi2 && !c->d_vobs) return fail(c, GLAD_ESTATE, "jam: chi2 requested but no vrms_obs/vrms_ivar set");
    if (!d_lum || !d_beta || (nm > 0 && !d_mass)) return fail(c, GLAD_EINVAL, "jam: null table pointer");
    if (nl <= 0 || nm < 0) return fail(c, GLAD_EINVAL, "jam: n_lum %d / n_mass %d", nl, nm);
    if (nl > GLAD_MAX_GAUSS || nm > GLAD_MAX_GAUSS) return fail(c, GLAD_ESHAPE, "jam: more than GLAD_MAX_GAUSS Gaussians");
    if (lum_stride < 0 || mass_stride < 0) return fail(c, GLAD_EINVAL, "jam: negative stride");
    const int nmx = nm + 1;
    int NG;
    if (jam_quad_geometry(c, &NG) < 0) return fail(c, GLAD_ESHAPE, "jam: sky grid too large");
    if (jam_post_smem_bytes(c->nxf, c->nyf, nl) > (size_t)glad_smem_dynamic_max(c))
        return fail(c, GLAD_ESHAPE, "jam: folded grid %dx%d with %d luminous Gaussians needs %zu bytes of shared memory in the binning kernel, limit %d",
                    c->nxf, c->nyf, nl, jam_post_smem_bytes(c->nxf, c->nyf, nl), glad_smem_dynamic_max(c));
    // K-slices: enough CTAs for >= 4 per SM when the batch is small
    long M = (long)c->nu * nmx * nl;
    int NCH = (int)((M + NG * JQ_MI - 1) / (NG * JQ_MI));
    int S = (4 * c->sm_count + B - 1) / B;
    if (S > 32) S = 32;
    if (S > NCH) S = NCH;
    if (S < 1) S = 1;
    if (c->jam_slices >= 1) S = c->jam_slices < NCH ? c->jam_slices : NCH;
    glad_status st = grow(c, &c->d_jam_tab, &c->jam_tab_cap, (size_t)B * jam_table_floats(nl, nmx));
    if (st != GLAD_OK) return st;
    st = grow(c, &c->d_partial, &c->partial_cap, (size_t)B * S * c->nxf * c->nyf);
    if (st != GLAD_OK) return st;
    CU(launch_jam_prep(c, d_dyn, B, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta, per_gaussian), "jam_prep_kernel");
    if (!c->jam_simt && jam_quad_tc_supported(c, nl, nmx)) CU(launch_jam_quad_tc(c, B, nl, nmx, S), "jam_quad_tc_kernel");
    else CU(launch_jam_quad(c, B, nl, nmx, S), "jam_quad_kernel");
    CU(launch_jam_post(c, B, nl, nmx, S, d_vrms, d_chi2, d_v2map, d_flags), "jam_post_kernel");
    return GLAD_OK;
}

extern "C" {

glad_status glad_lens_image_batch(glad_ctx* c, const float* d_lens, int B, float* d_images, float* d_chi2, int32_t* d_flags) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && !d_lens)) return fail(c, GLAD_EINVAL, "glad_lens_image_batch: B=%d / null params", B);
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    return lens_impl(c, d_lens, B, d_images, d_chi2, d_flags);
}

glad_status glad_lens_image_noalloc(glad_ctx* c, const float* d_lens, int B, float* d_images, float* d_chi2, int32_t* d_flags) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && !d_lens)) return fail(c, GLAD_EINVAL, "glad_lens_image_noalloc: B=%d / null params", B);
    if (B > GLAD_LENS_NOALLOC_MAX_B)
        return fail(c, GLAD_ESHAPE, "glad_lens_image_noalloc: batch of %d vectors, the static constants array holds %d (GLAD_LENS_NOALLOC_MAX_B): split the batch",
                    B, GLAD_LENS_NOALLOC_MAX_B);
    if (B == 0) return GLAD_OK;
    if (!c->d_lens_const_static) return fail(c, GLAD_ESTATE, "glad_lens_image_noalloc: the address of the static array could not be taken at glad_create");
    if (!c->have_image) return fail(c, GLAD_ESTATE, "glad_lens_image_noalloc: glad_set_image_data not called");
    if (c->d_lambda && B > c->n_lambda) return fail(c, GLAD_EINVAL, "glad_lens_image_noalloc: batch of %d vectors but the mass sheet has %d lambdas", B, c->n_lambda);
    if (c->d_enfw && B > c->n_enfw) return fail(c, GLAD_EINVAL, "glad_lens_image_noalloc: batch of %d vectors but %d eNFW halos", B, c->n_enfw);
    if (d_chi2 && !c->d_data) return fail(c, GLAD_ESTATE, "glad_lens_image_noalloc: chi2 requested but no data/ivar set");
    DeviceScope ds(c);
    CU(launch_lens_noalloc(c, d_lens, B, d_images, d_chi2, d_flags), "lens kernels (static constants)");
    return GLAD_OK;
}

glad_status glad_jam_vrms_batch(glad_ctx* c, const float* d_dyn, int B, const float* d_lum, int nl, long lum_stride,
                                const float* d_mass, int nm, long mass_stride, const float* d_beta, int per_gaussian,
                                float* d_vrms, float* d_chi2, float* d_v2map, int32_t* d_flags) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && !d_dyn)) return fail(c, GLAD_EINVAL, "glad_jam_vrms_batch: B=%d / null params", B);
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    return jam_impl(c, d_dyn, B, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta, per_gaussian, d_vrms, d_chi2,
                    d_v2map, d_flags);
}

}  // extern "C"

extern "C" {

glad_status glad_set_jam_sph_rules(glad_ctx* c, const float* d_rgrid, int nr, const float* d_thgrid, int nth, const float* d_tau,
                                   const float* d_wtau, int nt, const float* d_un, const float* d_uw, int nu, const float* d_zeta,
                                   const float* d_wz, int nz) {
    if (!c) return GLAD_EINVAL;
    if (!d_rgrid) { c->have_sph = false; return GLAD_OK; }
    if (!d_thgrid || !d_tau || !d_wtau || !d_un || !d_uw || !d_zeta || !d_wz) return fail(c, GLAD_EINVAL, "glad_set_jam_sph_rules: null pointer");
    if (nr < 1 || nth < 1 || nt < 1 || nu < 1 || nz < 1) return fail(c, GLAD_EINVAL, "glad_set_jam_sph_rules: bad sizes");
    if (nr > GLAD_MAX_SPH_R || nth > GLAD_MAX_SPH_TH || nt > GLAD_MAX_NODES || nu > GLAD_MAX_NODES || nz > GLAD_MAX_NODES)
        return fail(c, GLAD_ESHAPE, "glad_set_jam_sph_rules: polar grid %d x %d / rules %d, %d, %d exceed the limits", nr, nth, nt, nu, nz);
    c->d_sph_r = d_rgrid; c->sph_nr = nr; c->d_sph_th = d_thgrid; c->sph_nth = nth;
    c->d_sph_tau = d_tau; c->d_sph_wtau = d_wtau; c->sph_nt = nt;
    c->d_sph_un = d_un; c->d_sph_uw = d_uw; c->sph_nu = nu;
    c->d_sph_zeta = d_zeta; c->d_sph_wz = d_wz; c->sph_nz = nz;
    c->have_sph = true;
    return GLAD_OK;
}

glad_status glad_jam_sph_vrms_batch(glad_ctx* c, const float* d_dyn, int B, const float* d_lum, int nl, long lum_stride,
                                    const float* d_mass, int nm, long mass_stride, const float* d_beta, int per_gaussian,
                                    float* d_vrms, float* d_chi2, float* d_v2map, float* d_moments, int32_t* d_flags) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && !d_dyn)) return fail(c, GLAD_EINVAL, "glad_jam_sph_vrms_batch: B=%d / null params", B);
    if (!c->have_kin) return fail(c, GLAD_ESTATE, "glad_jam_sph_vrms_batch: glad_set_kin_data not called");
    if (!c->have_sph) return fail(c, GLAD_ESTATE, "glad_jam_sph_vrms_batch: glad_set_jam_sph_rules not called");
    if (d_chi2 && !c->d_vobs) return fail(c, GLAD_ESTATE, "glad_jam_sph_vrms_batch: chi2 requested but no vrms_obs/vrms_ivar set");
    if (!d_lum || !d_beta || (nm > 0 && !d_mass)) return fail(c, GLAD_EINVAL, "glad_jam_sph_vrms_batch: null table pointer");
    if (nl <= 0 || nm < 0) return fail(c, GLAD_EINVAL, "glad_jam_sph_vrms_batch: n_lum %d / n_mass %d", nl, nm);
    if (nl > GLAD_MAX_GAUSS || nm > GLAD_MAX_GAUSS) return fail(c, GLAD_ESHAPE, "glad_jam_sph_vrms_batch: more than GLAD_MAX_GAUSS Gaussians");
    if (lum_stride < 0 || mass_stride < 0) return fail(c, GLAD_EINVAL, "glad_jam_sph_vrms_batch: negative stride");
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    const int nmx = nm + 1;
    if (!jam_sph_supported(c, nl, nmx))
        return fail(c, GLAD_ESHAPE, "glad_jam_sph_vrms_batch: the potential table of %d mass Gaussians x %d u-nodes does not fit shared memory", nmx, c->sph_nu);
    if (jam_post_smem_bytes(c->nxf, c->nyf, nl) > (size_t)glad_smem_dynamic_max(c))
        return fail(c, GLAD_ESHAPE, "glad_jam_sph_vrms_batch: folded grid %dx%d with %d luminous Gaussians does not fit the binning kernel", c->nxf, c->nyf, nl);
    glad_status st = grow(c, &c->d_jam_tab, &c->jam_tab_cap, (size_t)B * jam_table_floats(nl, nmx));
    if (st != GLAD_OK) return st;
    st = grow(c, &c->d_sph_tab, &c->sph_tab_cap, (size_t)B * jam_sph_table_floats(nl, nmx, c->sph_nu));
    if (st != GLAD_OK) return st;
    st = grow(c, &c->d_partial, &c->partial_cap, (size_t)B * c->nxf * c->nyf);
    if (st != GLAD_OK) return st;
    float* rat = d_moments;
    if (!rat) {
        st = grow(c, &c->d_sph_rat, &c->sph_rat_cap, (size_t)B * 3 * c->sph_nr * c->sph_nth);
        if (st != GLAD_OK) return st;
        rat = c->d_sph_rat;
    }
    CU(launch_jam_prep(c, d_dyn, B, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta, per_gaussian), "jam_prep_kernel");
    CU(launch_jam_sph(c, d_dyn, B, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta, per_gaussian, rat), "jam_sph kernels");
    CU(launch_jam_post(c, B, nl, nmx, 1, d_vrms, d_chi2, d_v2map, d_flags, 1.f), "jam_post_kernel");
    return GLAD_OK;
}

}  // extern "C"

// Both halves (and, with d_ddt, the quasar terms of Eq. 35-36 on the lens stream) followed by joint_kernel.
static glad_status joint_impl(glad_ctx* c, const float* d_lens, const float* d_dyn, int B, const float* d_lum, int nl,
                              long lum_stride, const float* d_mass, int nm, long mass_stride, const float* d_beta,
                              int per_gaussian, float* d_loglike, float* d_chi2_lens, float* d_chi2_dyn, int32_t* d_flags,
                              const float* d_ddt, float* d_chi2_img, float* d_chi2_tmd) {
    glad_status st = grow(c, &c->d_tmp, &c->tmp_cap, (size_t)2 * B);
    if (st != GLAD_OK) return st;
    st = grow(c, &c->d_tmpflags, &c->tmpflags_cap, (size_t)2 * B);
    if (st != GLAD_OK) return st;
    float* c2l = d_chi2_lens ? d_chi2_lens : c->d_tmp;
    float* c2d = d_chi2_dyn ? d_chi2_dyn : c->d_tmp + B;
    int32_t *fl = c->d_tmpflags, *fd = c->d_tmpflags + B;
    // scratch of both halves is grown before the fork (grow() may synchronise and free)
    st = grow(c, &c->d_lens_const, &c->lens_const_cap, (size_t)B * LC_SIZE);
    if (st != GLAD_OK) return st;
    float *c2i = nullptr, *c2t = nullptr;
    if (d_ddt) {
        st = grow(c, &c->d_qtmp, &c->qtmp_cap, (size_t)2 * B);
        if (st != GLAD_OK) return st;
        c2i = d_chi2_img ? d_chi2_img : c->d_qtmp;
        c2t = d_chi2_tmd ? d_chi2_tmd : c->d_qtmp + B;
    }
    if (c->overlap) {
        // fork: the lens half (lens_prep's serial b_n roots, then lens_image) runs on the side stream beside jam_prep /
        // jam_quad; both wait for everything enqueued so far, and the caller's stream waits for the lens half below
        CU(cudaEventRecord(c->ev_fork, c->stream), "fork");
        CU(cudaStreamWaitEvent(c->side_stream, c->ev_fork, 0), "fork");
        c->lens_stream = c->side_stream;
    }
    st = lens_impl(c, d_lens, B, nullptr, c2l, fl);
    if (st == GLAD_OK && d_ddt) {
        cudaError_t qe = launch_quasar(c, c->lens_stream, d_lens, d_ddt, B, c2i, c2t, nullptr, nullptr, nullptr);
        if (qe != cudaSuccess) st = cuda_fail(c, qe, "quasar_kernel");
    }
    c->lens_stream = c->stream;
    if (c->overlap) cudaEventRecord(c->ev_join, c->side_stream);
    glad_status st2 = st == GLAD_OK ? jam_impl(c, d_dyn, B, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta, per_gaussian,
                                               nullptr, c2d, nullptr, fd) : st;
    if (c->overlap) cudaStreamWaitEvent(c->stream, c->ev_join, 0);   // join, also when a half failed: nothing left dangling
    if (st2 != GLAD_OK) return st2;
    CU(launch_joint(c, B, c2l, c2d, c2i, c2t, fl, fd, d_loglike, d_flags), "joint_kernel");
    return GLAD_OK;
}

extern "C" {

glad_status glad_joint_loglike_batch(glad_ctx* c, const float* d_lens, const float* d_dyn, int B, const float* d_lum, int nl,
                                     long lum_stride, const float* d_mass, int nm, long mass_stride, const float* d_beta,
                                     int per_gaussian, float* d_loglike, float* d_chi2_lens, float* d_chi2_dyn,
                                     int32_t* d_flags) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && (!d_lens || !d_dyn || !d_loglike))) return fail(c, GLAD_EINVAL, "glad_joint_loglike_batch: B=%d / null pointer", B);
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    return joint_impl(c, d_lens, d_dyn, B, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta, per_gaussian, d_loglike,
                      d_chi2_lens, d_chi2_dyn, d_flags, nullptr, nullptr, nullptr);
}

glad_status glad_set_quasar_data(glad_ctx* c, int n_img, const double* h_theta, const double* h_sigma_theta, int ref_image,
                                 const double* h_dt_obs, const double* h_sigma_dt) {
    if (!c) return GLAD_EINVAL;
    if (n_img == 0) { c->have_qso = false; return GLAD_OK; }
    if (n_img < 0 || n_img > GLAD_MAX_QIMG) return fail(c, GLAD_ESHAPE, "glad_set_quasar_data: n_img %d outside [0, GLAD_MAX_QIMG]", n_img);
    if (!h_theta || !h_sigma_theta) return fail(c, GLAD_EINVAL, "glad_set_quasar_data: null positions");
    if (ref_image < 0 || ref_image >= n_img) return fail(c, GLAD_EINVAL, "glad_set_quasar_data: reference image %d", ref_image);
    if ((h_dt_obs == nullptr) != (h_sigma_dt == nullptr)) return fail(c, GLAD_EINVAL, "glad_set_quasar_data: dt_obs and sigma_dt go together");
    glad_quasar_data q;
    memset(&q, 0, sizeof(q));
    q.n_img = n_img;
    q.ref = ref_image;
    for (int i = 0; i < n_img; ++i) {
        if (!(h_sigma_theta[i] > 0.0)) return fail(c, GLAD_EINVAL, "glad_set_quasar_data: sigma_theta[%d] = %g", i, h_sigma_theta[i]);
        q.theta[2 * i] = h_theta[2 * i];
        q.theta[2 * i + 1] = h_theta[2 * i + 1];
        q.ivar_theta[i] = 1.0 / (h_sigma_theta[i] * h_sigma_theta[i]);
        if (h_dt_obs && i != ref_image && h_sigma_dt[i] > 0.0) {
            q.dt_obs[i] = h_dt_obs[i];
            q.ivar_dt[i] = 1.0 / (h_sigma_dt[i] * h_sigma_dt[i]);
        }
    }
    c->qso = q;
    c->have_qso = true;
    return GLAD_OK;
}

glad_status glad_quasar_chi2_batch(glad_ctx* c, const float* d_lens, const float* d_ddt, int B, float* d_chi2_img,
                                   float* d_chi2_tmd, double* d_theta_pre, double* d_dt_pre, double* d_beta) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && (!d_lens || !d_ddt))) return fail(c, GLAD_EINVAL, "glad_quasar_chi2_batch: B=%d / null pointer", B);
    if (!c->have_qso) return fail(c, GLAD_ESTATE, "glad_quasar_chi2_batch: glad_set_quasar_data not called");
    if (c->d_lambda && B > c->n_lambda) return fail(c, GLAD_EINVAL, "glad_quasar_chi2_batch: batch of %d vectors but the mass sheet has %d lambdas", B, c->n_lambda);
    if (c->d_enfw && B > c->n_enfw) return fail(c, GLAD_EINVAL, "glad_quasar_chi2_batch: batch of %d vectors but %d eNFW halos", B, c->n_enfw);
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    CU(launch_quasar(c, c->stream, d_lens, d_ddt, B, d_chi2_img, d_chi2_tmd, d_theta_pre, d_dt_pre, d_beta), "quasar_kernel");
    return GLAD_OK;
}

static glad_status pixsrc_impl(glad_ctx* c, const char* who, const float* d_lens, const float* d_src_grid, const float* d_lam, double lam_lo,
                               double lam_hi, float* d_lam_hat, int nsx, int nsy, int B, int scratch_mib_max, float* d_logev, float* d_chi2,
                               float* d_reg, float* d_s_mp, float* d_model, int32_t* d_flags) {
    const bool search = d_lam == nullptr;
    if (!c->have_image || !c->d_data || !c->d_ivar) return fail(c, GLAD_ESTATE, "%s: glad_set_image_data (with data and ivar) not called", who);
    if (c->d_enfw) return fail(c, GLAD_ESTATE, "%s: the eNFW halo is not part of this entry; clear it with glad_set_enfw(ctx, NULL, ...)", who);
    if (nsx < 2 || nsy < 2 || (long)nsx * nsy > 4096) return fail(c, GLAD_ESHAPE, "%s: source grid %d x %d (need >= 2 x 2, N_s <= 4096)", who, nsx, nsy);
    if (c->d_lambda && B > c->n_lambda) return fail(c, GLAD_EINVAL, "%s: batch of %d vectors but the mass sheet has %d lambdas", who, B, c->n_lambda);
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    const int npix = c->grid.nx * c->grid.ny, ns = nsx * nsy;
    const size_t cap = (size_t)(scratch_mib_max > 0 ? scratch_mib_max : 16384) << 20;
    const size_t one = pixsrc_scratch_bytes(npix, ns, 1, search);
    if (one > cap) return fail(c, GLAD_ESHAPE, "%s: one vector needs %zu bytes of scratch, limit %zu", who, one, cap);
    int Bc = (int)(cap / one);
    if (Bc > B) Bc = B;
    if (Bc > 2 * c->sm_count) Bc = 2 * c->sm_count;
    while (Bc > 1 && pixsrc_scratch_bytes(npix, ns, Bc, search) > cap) --Bc;
    Bc = (B + (B + Bc - 1) / Bc - 1) / ((B + Bc - 1) / Bc);   // equal chunks: a short tail chunk pays every launch latency again
    glad_status st = grow(c, &c->d_pix, &c->pix_cap, pixsrc_scratch_bytes(npix, ns, Bc, search), true);
    if (st != GLAD_OK) return st;
    // ln det g in closed form: g = kron(I, T^2) + kron(T^2, I), T the (1,-2,1) matrix with eigenvalues -2 + 2 cos(k pi/(n+1))
    double logdet_g = 0.0;
    for (int j = 1; j <= nsy; ++j)
        for (int i = 1; i <= nsx; ++i) {
            const double mx = -2.0 + 2.0 * cos(i * M_PI / (nsx + 1)), my = -2.0 + 2.0 * cos(j * M_PI / (nsy + 1));
            logdet_g += log(mx * mx + my * my);
        }
    for (int b0 = 0; b0 < B; b0 += Bc) {
        const int nb = B - b0 < Bc ? B - b0 : Bc;
        CU(launch_pixsrc_chunk(c, c->d_pix, d_lens + (size_t)b0 * GLAD_NLENS, d_src_grid + (size_t)b0 * 3, d_lam ? d_lam + b0 : nullptr,
                               c->d_lambda ? c->d_lambda + b0 : nullptr, nsx, nsy, nb, logdet_g, d_logev ? d_logev + b0 : nullptr,
                               d_chi2 ? d_chi2 + b0 : nullptr, d_reg ? d_reg + b0 : nullptr,
                               d_s_mp ? d_s_mp + (size_t)b0 * ns : nullptr, d_model ? d_model + (size_t)b0 * npix : nullptr,
                               d_flags ? d_flags + b0 : nullptr, lam_lo, lam_hi, d_lam_hat ? d_lam_hat + b0 : nullptr),
           "pixsrc kernels");
    }
    return GLAD_OK;
}

glad_status glad_pixsrc_evidence_batch(glad_ctx* c, const float* d_lens, const float* d_src_grid, const float* d_lam, int nsx, int nsy,
                                       int B, int scratch_mib_max, float* d_logev, float* d_chi2, float* d_reg, float* d_s_mp,
                                       float* d_model, int32_t* d_flags) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && (!d_lens || !d_src_grid || !d_lam))) return fail(c, GLAD_EINVAL, "glad_pixsrc_evidence_batch: B=%d / null pointer", B);
    return pixsrc_impl(c, "glad_pixsrc_evidence_batch", d_lens, d_src_grid, d_lam, 0.0, 0.0, nullptr, nsx, nsy, B, scratch_mib_max, d_logev, d_chi2,
                       d_reg, d_s_mp, d_model, d_flags);
}

glad_status glad_pixsrc_lambda_opt_batch(glad_ctx* c, const float* d_lens, const float* d_src_grid, float lam_lo, float lam_hi, int nsx, int nsy,
                                         int B, int scratch_mib_max, float* d_lam_hat, float* d_logev, float* d_chi2, float* d_reg,
                                         float* d_s_mp, float* d_model, int32_t* d_flags) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && (!d_lens || !d_src_grid || !d_lam_hat))) return fail(c, GLAD_EINVAL, "glad_pixsrc_lambda_opt_batch: B=%d / null pointer", B);
    if (!(lam_lo > 0.f) || !(lam_hi > lam_lo) || !isfinite(lam_hi)) return fail(c, GLAD_EINVAL, "glad_pixsrc_lambda_opt_batch: lambda range [%g, %g]", lam_lo, lam_hi);
    return pixsrc_impl(c, "glad_pixsrc_lambda_opt_batch", d_lens, d_src_grid, nullptr, (double)lam_lo, (double)lam_hi, d_lam_hat, nsx, nsy, B,
                       scratch_mib_max, d_logev, d_chi2, d_reg, d_s_mp, d_model, d_flags);
}

glad_status glad_joint_loglike_host(glad_ctx* c, const float* h_lens, const float* h_dyn, int B, const float* h_lum, int nl,
                                    long lum_stride, const float* h_mass, int nm, long mass_stride, const float* h_beta,
                                    int per_gaussian, float* h_loglike, float* h_chi2_lens, float* h_chi2_dyn,
                                    int32_t* h_flags) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && (!h_lens || !h_dyn || !h_loglike || !h_lum || !h_beta || (nm > 0 && !h_mass))))
        return fail(c, GLAD_EINVAL, "glad_joint_loglike_host: B=%d / null pointer", B);
    if (nl <= 0 || nm < 0 || lum_stride < 0 || mass_stride < 0) return fail(c, GLAD_EINVAL, "glad_joint_loglike_host: bad table sizes");
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    auto r4 = [](size_t n) { return (n + 3) & ~(size_t)3; };
    size_t n_lens = r4((size_t)B * GLAD_NLENS), n_dyn = r4((size_t)B * GLAD_NDYN);
    size_t n_lum = r4(lum_stride ? (size_t)B * lum_stride : (size_t)nl * 3);
    size_t n_mass = r4(mass_stride ? (size_t)B * mass_stride : (size_t)nm * 3);
    size_t n_beta = r4(per_gaussian ? (size_t)B * nl : (size_t)B), n_out = r4((size_t)B);
    glad_status st = grow(c, &c->d_stage, &c->stage_cap, n_lens + n_dyn + n_lum + n_mass + n_beta + 4 * n_out);
    if (st != GLAD_OK) return st;
    float* d_lens = c->d_stage;
    float* d_dyn = d_lens + n_lens;
    float* d_lum = d_dyn + n_dyn;
    float* d_mass = d_lum + n_lum;
    float* d_beta = d_mass + n_mass;
    float* d_ll = d_beta + n_beta;
    float* d_c2l = d_ll + n_out;
    float* d_c2d = d_c2l + n_out;
    int32_t* d_fl = (int32_t*)(d_c2d + n_out);
    cudaStream_t s = c->stream;
    CU(cudaMemcpyAsync(d_lens, h_lens, sizeof(float) * B * GLAD_NLENS, cudaMemcpyHostToDevice, s), "H2D lens");
    CU(cudaMemcpyAsync(d_dyn, h_dyn, sizeof(float) * B * GLAD_NDYN, cudaMemcpyHostToDevice, s), "H2D dyn");
    CU(cudaMemcpyAsync(d_lum, h_lum, sizeof(float) * (lum_stride ? (size_t)B * lum_stride : (size_t)nl * 3), cudaMemcpyHostToDevice, s), "H2D lum");
    if (nm > 0)
        CU(cudaMemcpyAsync(d_mass, h_mass, sizeof(float) * (mass_stride ? (size_t)B * mass_stride : (size_t)nm * 3), cudaMemcpyHostToDevice, s), "H2D mass");
    CU(cudaMemcpyAsync(d_beta, h_beta, sizeof(float) * (per_gaussian ? (size_t)B * nl : (size_t)B), cudaMemcpyHostToDevice, s), "H2D beta");
    st = glad_joint_loglike_batch(c, d_lens, d_dyn, B, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta, per_gaussian,
                                  d_ll, d_c2l, d_c2d, d_fl);
    if (st != GLAD_OK) return st;
    CU(cudaMemcpyAsync(h_loglike, d_ll, sizeof(float) * B, cudaMemcpyDeviceToHost, s), "D2H loglike");
    if (h_chi2_lens) CU(cudaMemcpyAsync(h_chi2_lens, d_c2l, sizeof(float) * B, cudaMemcpyDeviceToHost, s), "D2H chi2");
    if (h_chi2_dyn) CU(cudaMemcpyAsync(h_chi2_dyn, d_c2d, sizeof(float) * B, cudaMemcpyDeviceToHost, s), "D2H chi2");
    if (h_flags) CU(cudaMemcpyAsync(h_flags, d_fl, sizeof(int32_t) * B, cudaMemcpyDeviceToHost, s), "D2H flags");
    CU(cudaStreamSynchronize(s), "joint (host) sync");
    return GLAD_OK;
}

static glad_status mge_check(glad_ctx* c, const char* who, int n, float lo, float hi) {
    if (n < 2 || !(lo > 0.f) || !(hi > lo)) return fail(c, GLAD_EINVAL, "%s: n_gauss %d on [%g, %g]", who, n, lo, hi);
    if (n > GLAD_MAX_GAUSS) return fail(c, GLAD_ESHAPE, "%s: more than GLAD_MAX_GAUSS Gaussians", who);
    return GLAD_OK;
}
#define MGE_DEFAULT_ORDER 12

glad_status glad_mge1d_batch(glad_ctx* c, int kind, const float* d_prof, int B, int n_gauss, float sigma_lo, float sigma_hi,
                             int P, float* d_mge) {
    if (!c) return GLAD_EINVAL;
    if (B < 0 || (B > 0 && (!d_prof || !d_mge))) return fail(c, GLAD_EINVAL, "glad_mge1d_batch: B=%d / null pointer", B);
    if (kind != GLAD_PROFILE_SERSIC && kind != GLAD_PROFILE_EPL && kind != GLAD_PROFILE_CHAMELEON && kind != GLAD_PROFILE_NFW_CSE)
        return fail(c, GLAD_EINVAL, "glad_mge1d_batch: profile kind %d", kind);
    if (kind == GLAD_PROFILE_NFW_CSE && !c->d_cse64) return fail(c, GLAD_ESTATE, "glad_mge1d_batch: GLAD_PROFILE_NFW_CSE needs the CSE table of glad_set_enfw");
    if (P == 0) P = MGE_DEFAULT_ORDER;
    if (P < 1 || P > 15) return fail(c, GLAD_EINVAL, "glad_mge1d_batch: Euler order %d outside [1,15]", P);
    glad_status st = mge_check(c, "glad_mge1d_batch", n_gauss, sigma_lo, sigma_hi);
    if (st != GLAD_OK) return st;
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    CU(launch_mge1d(c, kind, d_prof, B, n_gauss, sigma_lo, sigma_hi, P, d_mge), "mge1d_kernel");
    return GLAD_OK;
}

}  // extern "C"

static glad_status model_impl(glad_ctx* c, const float* d_lens, const float* d_dyn, const float* d_ddt, float zd,
                              int B, int nl, float lum_lo, float lum_hi, int nm, float mass_lo, float mass_hi,
                              const float* d_beta, int per_gaussian, float* d_loglike, float* d_chi2_lens,
                              float* d_chi2_dyn, int32_t* d_flags, float* d_lum_out, float* d_mass_out, bool quasar,
                              float* d_chi2_img, float* d_chi2_tmd) {
    if (!c) return GLAD_EINVAL;
    if (quasar && !c->have_qso) return fail(c, GLAD_ESTATE, "glad_joint_loglike_full_batch: glad_set_quasar_data not called");
    if (B < 0 || (B > 0 && (!d_lens || !d_dyn || !d_ddt || !d_beta || !d_loglike)))
        return fail(c, GLAD_EINVAL, "glad_joint_loglike_model_batch: B=%d / null pointer", B);
    if (!(zd > -1.f)) return fail(c, GLAD_EINVAL, "glad_joint_loglike_model_batch: z_d = %g", zd);
    glad_status st = mge_check(c, "glad_joint_loglike_model_batch (luminous)", nl, lum_lo, lum_hi);
    if (st != GLAD_OK) return st;
    st = mge_check(c, "glad_joint_loglike_model_batch (mass)", nm, mass_lo, mass_hi);
    if (st != GLAD_OK) return st;
    if (B == 0) return GLAD_OK;
    DeviceScope ds(c);
    if (c->d_lambda && B > c->n_lambda) return fail(c, GLAD_EINVAL, "joint model: batch of %d vectors but the mass sheet has %d lambdas", B, c->n_lambda);
    if (c->d_enfw && B > c->n_enfw) return fail(c, GLAD_EINVAL, "joint model: batch of %d vectors but %d eNFW halos", B, c->n_enfw);
    const int nmt = nm + (c->d_lambda ? c->ms_n : 0) + (c->d_enfw ? c->nf_n : 0);      // the mass sheet and the halo add rows of their own
    if (nmt > GLAD_MAX_GAUSS) return fail(c, GLAD_ESHAPE, "joint model: n_mass %d + %d sheet Gaussians exceed GLAD_MAX_GAUSS", nm, nmt - nm);
    const size_t n_lens = (size_t)B * GLAD_NLENS, n_lum = (size_t)B * nl * 3, n_mass = (size_t)B * nmt * 3;
    st = grow(c, &c->d_model, &c->model_cap, n_lens + n_lum + n_mass);
    if (st != GLAD_OK) return st;
    float* m_lens = c->d_model;
    float* m_lum = d_lum_out ? d_lum_out : m_lens + n_lens;
    float* m_mass = d_mass_out ? d_mass_out : m_lens + n_lens + n_lum;
    CU(launch_model(c, d_lens, d_dyn, d_ddt, (double)zd, B, (c->light_kinds & 2) ? GLAD_PROFILE_CHAMELEON : GLAD_PROFILE_SERSIC, nl, lum_lo, lum_hi, nm, mass_lo, mass_hi, MGE_DEFAULT_ORDER, m_lens,
                    m_lum, m_mass), "model_kernel");
    return joint_impl(c, m_lens, d_dyn, B, m_lum, nl, 3L * nl, m_mass, nmt, 3L * nmt, d_beta, per_gaussian, d_loglike, d_chi2_lens,
                      d_chi2_dyn, d_flags, quasar ? d_ddt : nullptr, d_chi2_img, d_chi2_tmd);
}

extern "C" {

glad_status glad_joint_loglike_model_batch(glad_ctx* c, const float* d_lens, const float* d_dyn, const float* d_ddt, float zd,
                                           int B, int nl, float lum_lo, float lum_hi, int nm, float mass_lo, float mass_hi,
                                           const float* d_beta, int per_gaussian, float* d_loglike, float* d_chi2_lens,
                                           float* d_chi2_dyn, int32_t* d_flags, float* d_lum_out, float* d_mass_out) {
    return model_impl(c, d_lens, d_dyn, d_ddt, zd, B, nl, lum_lo, lum_hi, nm, mass_lo, mass_hi, d_beta, per_gaussian, d_loglike,
                      d_chi2_lens, d_chi2_dyn, d_flags, d_lum_out, d_mass_out, false, nullptr, nullptr);
}

glad_status glad_joint_loglike_full_batch(glad_ctx* c, const float* d_lens, const float* d_dyn, const float* d_ddt, float zd,
                                          int B, int nl, float lum_lo, float lum_hi, int nm, float mass_lo, float mass_hi,
                                          const float* d_beta, int per_gaussian, float* d_loglike, float* d_chi2_lens,
                                          float* d_chi2_dyn, float* d_chi2_img, float* d_chi2_tmd, int32_t* d_flags) {
    return model_impl(c, d_lens, d_dyn, d_ddt, zd, B, nl, lum_lo, lum_hi, nm, mass_lo, mass_hi, d_beta, per_gaussian, d_loglike,
                      d_chi2_lens, d_chi2_dyn, d_flags, nullptr, nullptr, true, d_chi2_img, d_chi2_tmd);
}

}  // extern "C"
