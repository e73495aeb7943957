// Dynamics half of libglad, everything except the quadrature kernel (jam_quad.cu):
//   jam_prep_kernel    rows a0/a5: deprojection (Eq. 22-25), BH Gaussian (R-D3), unit scale,
//                      per-Gaussian and per-pair constants in fp64 -> fp32 table block per vector.
//   kin_weights_kernel static: W[l][pf] = sum_{p in bin l} K(p - p') summed over the mirror images p' of the
//                      folded pixel pf.  Because PSF convolution and bin sums are linear, Eq. 27 becomes
//                      num_l = sum_pf W[l][pf] * (Sigma v2)[pf],  den_l = sum_pf W[l][pf] * Sigma[pf].
//   jam_post_kernel    rows a7-a8: sum the K-slices, Sigma map (Eq. 21), bin dot products, sqrt (Eq. 28),
//                      chi2_D (Eq. 32), optional unfolded map output.
//   joint_kernel       row a9.
#include <math.h>

#include "glad_internal.h"

#define LOG2E 1.4426950408889634
#define G_NEWTON 0.004301            // (km/s)^2 pc / Msun (R-D1)
#define SIGMA_BH_ARCSEC 0.01         // R-D3 (paper's central softening scale)

__global__ void __launch_bounds__(128) jam_prep_kernel(const float* __restrict__ dyn, int B,
                                                      const float* __restrict__ lum, int nl, long lum_stride,
                                                      const float* __restrict__ mass, int nm, long mass_stride,
                                                      const float* __restrict__ beta, int per_gaussian,
                                                      float* __restrict__ tab) {
    const int b = blockIdx.x, tid = threadIdx.x;
    const int nmx = nm + 1;
    float* T = tab + (size_t)b * jam_table_floats(nl, nmx);
    float* TL = T + JT_HDR;
    float* TM = TL + JL_COUNT * nl;
    float* TC = TM + JM_COUNT * nmx;
    float* TD = TC + nmx * nl;
    __shared__ double s_sq[GLAD_MAX_GAUSS];      // sigma_k^2 q_k^2
    __shared__ double s_bk[GLAD_MAX_GAUSS];
    __shared__ double s_qj2[GLAD_MAX_GAUSS + 1]; // q_j^2
    __shared__ double s_sj2[GLAD_MAX_GAUSS + 1];
    __shared__ int s_bad;
    if (tid == 0) s_bad = 0;
    __syncthreads();

    const double inc = dyn[b * GLAD_NDYN + 0], Dd = dyn[b * GLAD_NDYN + 1];
    const double Mbh = dyn[b * GLAD_NDYN + 2], ups = dyn[b * GLAD_NDYN + 3];
    const double ci = cos(inc), si = sin(inc), ci2 = ci * ci, si2 = si * si;
    const double pc = Dd * 3.14159265358979323846 / 0.648;   // pc per arcsec
    const float* lt = lum + (size_t)b * lum_stride;
    const float* mt = mass + (size_t)b * mass_stride;
    const bool has_bh = Mbh > 0.0;
    bool bad = !(Dd > 0.0) || !(Mbh >= 0.0) || !(si > 0.0);

    for (int k = tid; k < nl; k += blockDim.x) {
        double I0 = lt[3 * k], sg = lt[3 * k + 1], qp = lt[3 * k + 2];
        double bz = per_gaussian ? beta[(size_t)b * nl + k] : beta[b];
        double d = qp * qp - ci2;
        if (!(d > 0.0) || !(sg > 0.0) || !(qp > 0.0) || !(bz < 1.0)) { bad = true; d = 1.0; sg = 1.0; qp = 1.0; bz = 0.0; }
        double q = sqrt(d) / si, q2 = q * q, s2 = sg * sg;
        double nu = I0 * qp / (q * sg * sqrt(2.0 * 3.14159265358979323846));   // per pc^2 per arcsec
        double bk = 1.0 / (1.0 - bz);
        s_sq[k] = s2 * q2;
        s_bk[k] = bk;
        TL[JL_INVS2 * nl + k] = (float)(1.0 / s2);
        TL[JL_BKQ * nl + k] = (float)((1.0 - q2) / (s2 * q2));
        TL[JL_S0 * nl + k] = (float)(nu * s2 * q2 * (ci2 + bk * si2));
        TL[JL_D0 * nl + k] = (float)(1.0 - bk * q2);
        TL[JL_NKS * nl + k] = (float)(nu * si2);
        TL[JL_I0 * nl + k] = (float)I0;
        TL[JL_E1 * nl + k] = (float)(LOG2E / (2.0 * s2));
        TL[JL_E2 * nl + k] = (float)(LOG2E / (2.0 * s2 * qp * qp));
    }
    for (int j = tid; j < nmx; j += blockDim.x) {
        double S0, sg, qp;
        if (j < nm) { S0 = ups * (double)mt[3 * j]; sg = mt[3 * j + 1]; qp = mt[3 * j + 2]; }
        else {
            sg = SIGMA_BH_ARCSEC; qp = 1.0;
            double sp = sg * pc;
            S0 = has_bh ? Mbh / (2.0 * 3.14159265358979323846 * sp * sp) : 0.0;
        }
        double d = qp * qp - ci2;
        if (!(d > 0.0) || !(sg > 0.0) || !(qp > 0.0)) { bad = true; d = 1.0; sg = 1.0; qp = 1.0; }
        double q = sqrt(d) / si, s2 = sg * sg;
        double rho = S0 * qp / (q * sg * sqrt(2.0 * 3.14159265358979323846));
        s_qj2[j] = q * q;
        s_sj2[j] = s2;
        TM[JM_INVS2 * nmx + j] = (float)(1.0 / s2);
        TM[JM_OMQ2 * nmx + j] = (float)(1.0 - q * q);
        TM[JM_MJ * nmx + j] = (float)(q * rho);
    }
    if (bad) s_bad = 1;
    __syncthreads();
    for (int e = tid; e < nmx * nl; e += blockDim.x) {
        int j = e / nl, k = e - j * nl;
        double C = 1.0 - s_qj2[j] - s_sq[k] / s_sj2[j];
        TC[e] = (float)C;
        TD[e] = (float)((1.0 - s_bk[k]) * C + (1.0 - s_qj2[j]) * s_bk[k]);
    }
    if (tid == 0) {
        // V^2 = 4 pi^{3/2} G (pc/arcsec) Phi(arcsec units, densities per pc^2)
        T[JH_SCALE] = (float)(4.0 * pow(3.14159265358979323846, 1.5) * G_NEWTON * pc);
        T[JH_COS2I] = (float)ci2;
        T[JH_SIN2I] = (float)si2;
        T[JH_NM] = __int_as_float(has_bh ? nmx : nm);
        T[JH_VALID] = __int_as_float(s_bad ? 0 : 1);
    }
}

// ---------------------------------------------------------------------------------------------------
// static bin weights
// ---------------------------------------------------------------------------------------------------
__global__ void kin_weights_kernel(const int32_t* __restrict__ bin_id, const float* __restrict__ kern, int kk, int nx,
                                   int ny, int nxf, int nyf, const int* __restrict__ unfoldx,
                                   const int* __restrict__ unfoldy, int nbins, float* __restrict__ W) {
    // one thread per (bin l, folded pixel pf); fixed summation order -> deterministic
    int npf = nxf * nyf;
    long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (long)nbins * npf) return;
    int l = (int)(e / npf), pf = (int)(e - (long)l * npf);
    int fy = pf / nxf, fx = pf - fy * nxf;
    int c = kk / 2;
    float acc = 0.f;
    for (int my = 0; my < 2; ++my) {
        int sy = unfoldy[2 * fy + my];
        if (sy < 0) continue;
        for (int mx = 0; mx < 2; ++mx) {
            int sx = unfoldx[2 * fx + mx];
            if (sx < 0) continue;
            // source pixel p' = (sy,sx) contributes K[dy][dx] to target p = (sy + dy - c, sx + dx - c)
            for (int dy = 0; dy < kk; ++dy) {
                int ty = sy + dy - c;
                if (ty < 0 || ty >= ny) continue;
                for (int dx = 0; dx < kk; ++dx) {
                    int tx = sx + dx - c;
                    if (tx < 0 || tx >= nx) continue;
                    if (bin_id[ty * nx + tx] == l) acc += kern[dy * kk + dx];
                }
            }
        }
    }
    W[e] = acc;
}

cudaError_t launch_kin_weights(glad_ctx* c) {
    long n = (long)c->nbins * c->nxf * c->nyf;
    c->launches++;
    kin_weights_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(c->d_bin_id, c->d_kernel, c->kk, c->nx, c->ny,
                                                                         c->nxf, c->nyf, c->d_unfoldx, c->d_unfoldy,
                                                                         c->nbins, c->d_binw);
    return cudaGetLastError();
}

cudaError_t launch_jam_prep(glad_ctx* c, const float* d_dyn, int B, const float* d_lum, int nl, long lum_stride,
                            const float* d_mass, int nm, long mass_stride, const float* d_beta, int per_gaussian) {
    ProfScope ps(c, GK_JAM_PREP);
    jam_prep_kernel<<<B, 128, 0, c->stream>>>(d_dyn, B, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta,
                                             per_gaussian, c->d_jam_tab);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// post: K-slice sum, Sigma map, bins, chi2
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__global__ void __launch_bounds__(256) jam_post_kernel(const float* __restrict__ tab, int tabsz, int nl, int nmx,
                                                      const float* __restrict__ partial, int S, int nx, int ny,
                                                      int nxf, int nyf, const float* __restrict__ xf2,
                                                      const float* __restrict__ yf2, const int* __restrict__ foldx,
                                                      const int* __restrict__ foldy, const int* __restrict__ Wptr,
                                                      const float2* __restrict__ Wnz,
                                                      const int* __restrict__ bin_cnt, int nbins,
                                                      const float* __restrict__ vobs, const float* __restrict__ vivar,
                                                      float* __restrict__ vrms, float* __restrict__ chi2,
                                                      float* __restrict__ v2map, int32_t* __restrict__ flags,
                                                      float unit_scale) {
    extern __shared__ __align__(16) float sm[];
    const int b = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const int npf = nxf * nyf;
    float* v2f = sm;
    float* sbf = v2f + npf;
    float* ex = sbf + npf;          // [nl][nxf]
    float* ey = ex + nl * nxf;      // [nl][nyf]
    __shared__ float s_chi[8];
    __shared__ int s_badbin;
    const float* T = tab + (size_t)b * tabsz;
    const float* TL = T + JT_HDR;
    const bool valid = __float_as_int(T[JH_VALID]) != 0;
    const float qnan = __int_as_float(0x7fc00000), pinf = __int_as_float(0x7f800000);
    if (!valid) {
        if (vrms) for (int l = tid; l < nbins; l += nthr) vrms[(size_t)b * nbins + l] = qnan;
        if (v2map) for (int i = tid; i < nx * ny; i += nthr) v2map[(size_t)b * nx * ny + i] = qnan;
        if (tid == 0) {
            if (chi2) chi2[b] = pinf;
            if (flags) flags[b] = GLAD_FLAG_DYN_INVALID;
        }
        return;
    }
    if (tid == 0) s_badbin = 0;
    const float scale = unit_scale > 0.f ? unit_scale : T[JH_SCALE];   // JAM_sph maps arrive in final units
    const float* P = partial + (size_t)b * S * npf;
    for (int i = tid; i < npf; i += nthr) {
        float a = 0.f;
        for (int s = 0; s < S; ++s) a += P[(size_t)s * npf + i];
        v2f[i] = a * scale;
    }
    for (int e = tid; e < nl * nxf; e += nthr) { int k = e / nxf; ex[e] = ex2_approx(-TL[JL_E1 * nl + k] * xf2[e - k * nxf]); }
    for (int e = tid; e < nl * nyf; e += nthr) { int k = e / nyf; ey[e] = ex2_approx(-TL[JL_E2 * nl + k] * yf2[e - k * nyf]); }
    __syncthreads();
    for (int i = tid; i < npf; i += nthr) {       // Sigma(x',y') = sum_k I0_k exp(-(x'^2 + y'^2/q'^2)/(2 sigma^2)), Eq. 21
        int fy = i / nxf, fx = i - fy * nxf;
        float a = 0.f;
        for (int k = 0; k < nl; ++k) a = fmaf(TL[JL_I0 * nl + k] * ex[k * nxf + fx], ey[k * nyf + fy], a);
        sbf[i] = a;
    }
    __syncthreads();
    if (v2map)
        for (int i = tid; i < nx * ny; i += nthr) {
            int iy = i / nx, ix = i - iy * nx;
            v2map[(size_t)b * nx * ny + i] = v2f[foldy[iy] * nxf + foldx[ix]];
        }
    // bins: one warp per bin, lanes over the non-zero weights of its row (contiguous {pixel, weight} pairs -> coalesced 8-byte
    // loads; the kernel K is compact, so a bin touches ~1/5 of the folded map)
    float cpart = 0.f;
    const int nwarp = nthr >> 5;
    for (int l = warp; l < nbins; l += nwarp) {
        float num = 0.f, den = 0.f;
        const int e1 = Wptr[l + 1];
        for (int e = Wptr[l] + lane; e < e1; e += 32) {
            const float2 w = Wnz[e];
            const int i = __float_as_int(w.x);
            num = fmaf(w.y, v2f[i], num);
            den = fmaf(w.y, sbf[i], den);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            num += __shfl_xor_sync(0xffffffffu, num, o);
            den += __shfl_xor_sync(0xffffffffu, den, o);
        }
        if (lane == 0) {
            float v2 = (bin_cnt[l] > 0 && den > 0.f) ? num / den : qnan;
            float v = (v2 >= 0.f) ? sqrtf(v2) : qnan;
            if (!(v == v)) s_badbin = 1;
            if (vrms) vrms[(size_t)b * nbins + l] = v;
            if (chi2) { float r = vobs[l] - v; cpart = fmaf(vivar[l] * r, r, cpart); }
        }
    }
    if (lane == 0) s_chi[warp] = cpart;
    __syncthreads();
    if (tid == 0) {
        float c2 = 0.f;
        for (int w = 0; w < nwarp; ++w) c2 += s_chi[w];
        if (chi2) chi2[b] = s_badbin ? pinf : c2;
        if (flags) flags[b] = s_badbin ? GLAD_FLAG_BIN_INVALID : 0;
    }
}

size_t jam_post_smem_bytes(int nxf, int nyf, int nl) {
    return sizeof(float) * (2 * (size_t)nxf * nyf + (size_t)nl * (nxf + nyf));
}

cudaError_t launch_jam_post(glad_ctx* c, int B, int nl, int nmx, int S, float* d_vrms, float* d_chi2,
                            float* d_v2map, int32_t* d_flags, float unit_scale) {
    const size_t smem = jam_post_smem_bytes(c->nxf, c->nyf, nl);
    if (smem > (size_t)glad_smem_dynamic_max(c)) return cudaErrorInvalidConfiguration;   // glad_set_kin_data checks this up front
    cudaError_t e = smem_optin(c, jam_post_kernel);
    if (e != cudaSuccess) return e;
    ProfScope ps(c, GK_JAM_POST);
    jam_post_kernel<<<B, 256, smem, c->stream>>>(c->d_jam_tab, jam_table_floats(nl, nmx), nl, nmx, c->d_partial, S, c->nx,
                                                c->ny, c->nxf, c->nyf, c->d_xf2, c->d_yf2, c->d_foldx, c->d_foldy,
                                                c->d_binw_ptr, c->d_binw_nz, c->d_bin_cnt, c->nbins, c->d_vobs, c->d_vivar, d_vrms,
                                                d_chi2, d_v2map, d_flags, unit_scale);
    return cudaGetLastError();
}

// row a9: lnL = -(chi2_L + chi2_D [+ chi2_img + chi2_tmd])/2 (Eq. 52-53, R-J1); -inf where a half is invalid
__global__ void joint_kernel(int B, const float* __restrict__ c2l, const float* __restrict__ c2d,
                             const float* __restrict__ c2img, const float* __restrict__ c2tmd,
                             const int32_t* __restrict__ fl, const int32_t* __restrict__ fd,
                             float* __restrict__ loglike, int32_t* __restrict__ flags) {
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    double s = (double)c2l[b] + (double)c2d[b];
    if (c2img) s += (double)c2img[b];
    if (c2tmd) s += (double)c2tmd[b];
    int f = fl[b] | fd[b];
    loglike[b] = (f == 0 && isfinite(s)) ? (float)(-0.5 * s) : -__int_as_float(0x7f800000);
    if (flags) flags[b] = f;
}

cudaError_t launch_joint(glad_ctx* c, int B, const float* d_c2l, const float* d_c2d, const float* d_c2img, const float* d_c2tmd,
                         const int32_t* d_fl, const int32_t* d_fd, float* d_loglike, int32_t* d_flags) {
    ProfScope ps(c, GK_JOINT);
    joint_kernel<<<(B + 127) / 128, 128, 0, c->stream>>>(B, d_c2l, d_c2d, d_c2img, d_c2tmd, d_fl, d_fd, d_loglike, d_flags);
    return cudaGetLastError();
}
