// Pixelated-source extended-image likelihood of libglad for sm_100a (paper Eq. 37-43 P:269-304,
// Table 1): for every parameter vector
//   pixsrc_map_kernel    L   : ray-shoot every image pixel centre in fp64 (Eq. 33), bilinear weights on the vector's source grid;
//                              L is kept as its <= 4 non-zeros per row ({top-left source pixel, (fx, fy)}), never dense
//   pixsrc_blur_kernel   f = B L (Eq. 38): a warp per image pixel scatters PSF tap x bilinear weight into a shared-memory row
//                              of N_s floats and streams the row out (f [N_pix, N_s] fp32, the one large intermediate)
//   pixsrc_syrk_tc_kernel (pixsrc_syrk_tc.cu)  F = f^T C_d^-1 f (Eq. 41) + lambda g -> A (lower triangle, fp64 store) and
//                              D = f^T C_d^-1 d (Eq. 42): tcgen05 MMAs on two-term fp16 operands, 128 x 128 output tiles
//   chol_*_kernel (pixsrc_chol.cu)  A = L L^T in fp64, ln det A: three kernels per 64-wide panel over the whole batch
//   pixsrc_solve_kernel  s_MP = A^-1 D (Eq. 40) by forward / backward substitution, E_S = 1/2 s^T g s from its pixel definition
//   pixsrc_model_kernel  f s_MP (Eq. 37) and chi^2 = sum ivar (f s - d)^2, a warp per image pixel
//   pixsrc_final_kernel  the evidence of Eq. 43 (R-P5), flags
// Readings R-P1..5 are stated in DESIGN.md section 2.
#include <math.h>

#include "glad_internal.h"
#include "glad_mass_fp64.cuh"
#include "pixsrc_common.cuh"

#define PX_MAP_THREADS 128
#define PX_BLUR_WARPS 8
#define PX_NB 32           // block length of the substitutions
#define PX_CHOL_THREADS 256

__device__ __forceinline__ bool pixsrc_valid(const float* __restrict__ p, float lam, float ps) {
    return (p[2] >= 0.f) && (p[3] > 1.f && p[3] < 3.f) && (p[4] > 0.f && p[4] <= 1.f) && (p[8] >= 0.f) && (lam > 0.f) &&
           isfinite(lam) && (ps > 0.f) && isfinite(ps);
}

// ------------------------------------------------------------------------------------------------------------------
// L: one thread per image pixel
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(PX_MAP_THREADS) pixsrc_map_kernel(const float* __restrict__ lens, const float* __restrict__ src_grid,
                                                                    const float* __restrict__ lam_reg, const float* __restrict__ ms_lambda,
                                                                    double ms_rc, double ms_rt, glad_image_grid g, int nsx, int nsy,
                                                                    int* __restrict__ idx, float2* __restrict__ wgt) {
    const int b = blockIdx.y;
    const int npix = g.nx * g.ny;
    const float* p = lens + (size_t)b * GLAD_NLENS;
    __shared__ MassConst m;
    if (threadIdx.x == 0) {
        mass_const(p, ms_lambda ? (double)ms_lambda[b] : 1.0, ms_rc, ms_rt, ms_lambda != nullptr, m);
        mass_const_halo(nullptr, nullptr, 0, m);
    }
    __syncthreads();
    const int q = blockIdx.x * PX_MAP_THREADS + threadIdx.x;
    if (q >= npix) return;
    const float* sg = src_grid + (size_t)b * 3;
    int id = -1;
    float2 w = make_float2(0.f, 0.f);
    if (pixsrc_valid(p, lam_reg ? lam_reg[b] : 1.f, sg[2])) {     // lam_reg == NULL: lambda is searched for (Eq. 43)
        const int iy = q / g.nx, ix = q - iy * g.nx;
        const double thx = (double)g.x0 + ix * (double)g.pix, thy = (double)g.y0 + iy * (double)g.pix;
        MassEval e;
        mass_eval(m, thx, thy, e);
        const double tx = (thx - e.ax - (double)sg[0]) / (double)sg[2], ty = (thy - e.ay - (double)sg[1]) / (double)sg[2];
        if (isfinite(tx) && isfinite(ty) && tx >= 0.0 && ty >= 0.0 && tx < (double)(nsx - 1) && ty < (double)(nsy - 1)) {
            const int i0 = (int)floor(tx), j0 = (int)floor(ty);
            id = j0 * nsx + i0;
            w = make_float2((float)(tx - i0), (float)(ty - j0));
        }
    }
    idx[(size_t)b * npix + q] = id;
    wgt[(size_t)b * npix + q] = w;
}

// ------------------------------------------------------------------------------------------------------------------
// f = B L: a warp per image pixel, row in shared memory.  A row is non-zero only between the first and the last source pixel that the
// PSF footprint of its image pixel maps to (about a third of the row at the paper's sizes); the range goes to rng, which
// pixsrc_model_kernel uses to read only that part and pixsrc_syrk_tc_kernel to list the rows that count for a tile.  (Writing only
// the range and letting the contraction zero-fill the rest while it stages was measured: the kernel is bound by its shared-memory
// atomics, not by its stores -- 10.6 -> 10.1 ms -- and the range test cost the contraction 1.6 ms.)
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32 * PX_BLUR_WARPS) pixsrc_blur_kernel(const int* __restrict__ idx, const float2* __restrict__ wgt,
                                                                         const float* __restrict__ psf, int kpsf, int nx, int ny,
                                                                         int nsx, int ns, int rows_per_cta, float* __restrict__ f,
                                                                         int2* __restrict__ rng, const double* __restrict__ stat) {
    // The row is accumulated in 32-bit FIXED POINT: a float atomicAdd on shared memory is a compare-and-swap loop on this
    // architecture (LDS, FADD, ATOMS.CAST.SPIN, branch; retried when lanes collide, and neighbouring image pixels map into the
    // same source cell), an int atomicAdd is one ATOMS.ADD.  |f| <= sum |psf| =: S (bilinear weights sum to 1), so the scale
    // 2^30 / S cannot overflow; each of the <= K^2 terms is rounded to S 2^-31: |error| <= K^2 S 2^-31 (2e-7 S for a 21 x 21 PSF,
    // at the level of the 22-bit operands the contraction makes of f).  Measured: 10.5 -> 5.2 ms per 296 vectors at N_s = 1024; a
    // second word per entry that carries the remainders in units of S 2^-50 (f then exact to fp32 rounding; 9.9 ms) gives the same
    // errors against the fp64 definition in the parity tests (ln evidence 4.9e-8 on C2 32 x 32; 1.6e-5 on the ill-conditioned C1 32 x 20 case, float atomics 9e-6:
    // the contraction's operands, not this rounding, set them), so one word is kept.
    extern __shared__ int px_rows[];
    const int b = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int npix = nx * ny, cc = kpsf / 2, k2 = kpsf * kpsf;
    int* row = px_rows + (size_t)warp * ns;
    const float S = (float)stat[3];
    const float fx = S > 0.f ? 1073741824.f / S : 0.f, ifx = S > 0.f ? S / 1073741824.f : 0.f;
    const int* ib = idx + (size_t)b * npix;
    const float2* wb = wgt + (size_t)b * npix;
    const int p0 = blockIdx.x * rows_per_cta;
    for (int i = lane; i < ns; i += 32) row[i] = 0;        // the row is all zero between pixels: the written range is cleared after use
    __syncwarp();
    const int sdy = 32 / kpsf, sdx = 32 - sdy * kpsf;
    for (int r = warp; r < rows_per_cta; r += PX_BLUR_WARPS) {
        const int p = p0 + r;
        if (p >= npix) break;
        const int iy = p / nx, ix = p - iy * nx;
        int lo = 0x7fffffff, hi = -1;             // first and last source pixel this row touches (row-major index)
        // tap t = lane, lane + 32, ..: (dy, dx) is carried, not divided (32 = sdy * kpsf + sdx)
        int dy = lane / kpsf, dx = lane - dy * kpsf;
        for (int t = lane; t < k2; t += 32, dy += sdy, dx += sdx) {
            if (dx >= kpsf) { dx -= kpsf; ++dy; }
            const int sy = iy - (dy - cc), sx = ix - (dx - cc);
            if (sy < 0 || sy >= ny || sx < 0 || sx >= nx) continue;
            const int q = sy * nx + sx;
            const int id = ib[q];
            if (id < 0) continue;
            const float2 w = wb[q];
            const float a = psf[t] * fx;
            const float ax0 = a * (1.f - w.x), ax1 = a * w.x;
            atomicAdd(&row[id], __float2int_rn(ax0 * (1.f - w.y)));
            atomicAdd(&row[id + 1], __float2int_rn(ax1 * (1.f - w.y)));
            atomicAdd(&row[id + nsx], __float2int_rn(ax0 * w.y));
            atomicAdd(&row[id + nsx + 1], __float2int_rn(ax1 * w.y));
            lo = min(lo, id);
            hi = max(hi, id + nsx + 1);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        if (lane == 0) rng[(size_t)b * npix + p] = make_int2(lo, hi);
        __syncwarp();
        float* out = f + ((size_t)b * npix + p) * ns;
        for (int i = lane; i < ns; i += 32) out[i] = (float)row[i] * ifx;
        if (hi >= 0)
            for (int i = lo + lane; i <= hi; i += 32) row[i] = 0;
        __syncwarp();
    }
}

// F = f^T C_d^-1 f (+ lambda g) and D = f^T C_d^-1 d: pixsrc_syrk_tc.cu (tcgen05)

// ------------------------------------------------------------------------------------------------------------------
// Solve with the factor of pixsrc_chol.cu, regulariser: one CTA per vector, fp64
// ------------------------------------------------------------------------------------------------------------------
// out[b*PX_OUT + {0,1,2,3,4}] = {ln det A (chol_diag_kernel), E_S, chi2 (filled by pixsrc_model_kernel), not-positive-definite flag
// (chol_diag_kernel), y^T y = D^T A^-1 D}
// search = 1 (the lambda_hat search of Eq. 43): stop after the forward substitution -- the objective needs ln det A and y^T y only
#define PX_OUT 6
__global__ void __launch_bounds__(PX_CHOL_THREADS, 2) pixsrc_solve_kernel(const double* __restrict__ A, const double* __restrict__ D, int ns,
                                                                       int nsx, int nsy, double* __restrict__ s_out,
                                                                       double* __restrict__ out, int search) {
    extern __shared__ double px_sm[];
    double* yv = px_sm;                          // [ns]
    double* red = yv + ns;                       // [8][32]
    double* blk = red + (PX_CHOL_THREADS / 32) * 32;   // [32][33]: the diagonal block of the step (its serial part reads shared memory)
    const int b = blockIdx.x, tid = threadIdx.x;
    const double* Ab = A + (size_t)b * ns * ns;

    // forward substitution L y = D
    const int warp = tid >> 5, lane = tid & 31;
    const double* Db = D + (size_t)b * ns;
    for (int k0 = 0; k0 < ns; k0 += PX_NB) {
        const int nb = min(PX_NB, ns - k0);
        for (int r = warp; r < nb; r += PX_CHOL_THREADS / 32) {
            const double* lrow = Ab + (size_t)(k0 + r) * ns;
            double v = 0.0;
            for (int c = lane; c < k0; c += 32) v += lrow[c] * yv[c];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) yv[k0 + r] = Db[k0 + r] - v;
        }
        for (int e = tid; e < PX_NB * PX_NB; e += PX_CHOL_THREADS) {
            const int r = e >> 5, cc = e & 31;
            blk[r * (PX_NB + 1) + cc] = (r < nb && cc <= r) ? Ab[(size_t)(k0 + r) * ns + k0 + cc] : 0.0;
        }
        __syncthreads();
        if (warp == 0) {
            for (int r = 0; r < nb; ++r) {
                const double* lrow = blk + r * (PX_NB + 1);
                double v = (lane < r) ? lrow[lane] * yv[k0 + lane] : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0) yv[k0 + r] = (yv[k0 + r] - v) / lrow[r];
                __syncwarp();
            }
        }
        __syncthreads();
    }
    if (search) {
        double yy = 0.0;
        for (int a = tid; a < ns; a += PX_CHOL_THREADS) yy += yv[a] * yv[a];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) yy += __shfl_xor_sync(0xffffffffu, yy, o);
        if (lane == 0) red[warp] = yy;
        __syncthreads();
        if (tid == 0) {
            double t = 0.0;
            for (int w = 0; w < PX_CHOL_THREADS / 32; ++w) t += red[w];
            out[(size_t)b * PX_OUT + 4] = t;
        }
        return;
    }
    // backward substitution L^T s = y (s overwrites yv from the end)
    const int nblk = (ns + PX_NB - 1) / PX_NB;
    for (int kb = nblk - 1; kb >= 0; --kb) {
        const int k0 = kb * PX_NB, nb = min(PX_NB, ns - k0);
        // t_c = sum_{r >= k0 + nb} L[r, k0 + c] s_r : 8 row groups x 32 columns
        double v = 0.0;
        if (lane < nb)
            for (int r = k0 + nb + warp; r < ns; r += PX_CHOL_THREADS / 32) v += Ab[(size_t)r * ns + k0 + lane] * yv[r];
        red[warp * 32 + lane] = v;
        for (int e = tid; e < PX_NB * PX_NB; e += PX_CHOL_THREADS) {
            const int r = e >> 5, cc = e & 31;
            blk[r * (PX_NB + 1) + cc] = (r < nb && cc <= r) ? Ab[(size_t)(k0 + r) * ns + k0 + cc] : 0.0;
        }
        __syncthreads();
        if (warp == 0) {
            double t = 0.0;
#pragma unroll
            for (int g2 = 0; g2 < PX_CHOL_THREADS / 32; ++g2) t += red[g2 * 32 + lane];
            if (lane < nb) yv[k0 + lane] -= t;
            __syncwarp();
            for (int c = nb - 1; c >= 0; --c) {
                // s_c = (y_c - sum_{r in block, r > c} L[k0 + r, k0 + c] s_r) / L[c, c]
                double u = (lane > c && lane < nb) ? blk[lane * (PX_NB + 1) + c] * yv[k0 + lane] : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) u += __shfl_xor_sync(0xffffffffu, u, o);
                if (lane == 0) yv[k0 + c] = (yv[k0 + c] - u) / blk[c * (PX_NB + 1) + c];
                __syncwarp();
            }
        }
        __syncthreads();
    }
    // E_S = 1/2 sum_pixels [(s_{i-1} - 2 s_i + s_{i+1})^2 + (s_{j-1} - 2 s_j + s_{j+1})^2], s = 0 outside (R-P3)
    double es = 0.0;
    for (int a = tid; a < ns; a += PX_CHOL_THREADS) {
        const int j = a / nsx, i = a - j * nsx;
        const double s0 = yv[a];
        const double dx = (i > 0 ? yv[a - 1] : 0.0) - 2.0 * s0 + (i < nsx - 1 ? yv[a + 1] : 0.0);
        const double dy = (j > 0 ? yv[a - nsx] : 0.0) - 2.0 * s0 + (j < nsy - 1 ? yv[a + nsx] : 0.0);
        es += 0.5 * (dx * dx + dy * dy);
        s_out[(size_t)b * ns + a] = s0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) es += __shfl_xor_sync(0xffffffffu, es, o);
    __syncthreads();
    if (lane == 0) red[warp] = es;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int w = 0; w < PX_CHOL_THREADS / 32; ++w) t += red[w];
        out[(size_t)b * PX_OUT + 1] = t;
    }
}

// model = f s, chi2 = sum ivar (model - d)^2 : a warp per image pixel, 64 pixels per CTA
__global__ void __launch_bounds__(256) pixsrc_model_kernel(const float* __restrict__ f, const double* __restrict__ s,
                                                           const float* __restrict__ ivar, const float* __restrict__ data, int npix,
                                                           int ns, float* __restrict__ model, long model_stride,
                                                           double* __restrict__ out, const int2* __restrict__ rng) {
    extern __shared__ double px_s[];
    const int b = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < ns; i += 256) px_s[i] = s[(size_t)b * ns + i];
    __syncthreads();
    double c2 = 0.0;
    const int per = 64;
    for (int r = warp; r < per; r += 8) {
        const int p = blockIdx.x * per + r;
        if (p >= npix) break;
        const float* row = f + ((size_t)b * npix + p) * ns;
        double v = 0.0;
        const int2 rg = rng[(size_t)b * npix + p];                     // the row is zero outside its range
        if (rg.y >= 0)
            for (int i = (rg.x & ~3) + lane, i1 = min(rg.y | 3, ns - 1); i <= i1; i += 32) v += (double)row[i] * px_s[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) {
            if (model) model[(size_t)b * model_stride + p] = (float)v;
            const double w = (double)ivar[p];
            if (w != 0.0) { const double rr = v - (double)data[p]; c2 += w * rr * rr; }
        }
    }
    if (lane == 0 && c2 != 0.0) atomicAdd(&out[(size_t)b * PX_OUT + 2], c2);
}

// N_d and sum ln ivar over the unmasked pixels, max ivar and sum |psf| (the operand scales of the tensor-core contraction): static
// data; one CTA.  st[0..3]
__global__ void __launch_bounds__(256) pixsrc_static_kernel(const float* __restrict__ ivar, int npix, const float* __restrict__ psf,
                                                            int ktaps, double* __restrict__ st) {
    __shared__ double r1[256], r2[256], r3[256], r4[256];
    double n = 0.0, sl = 0.0, wm = 0.0, ps = 0.0;
    for (int p = threadIdx.x; p < npix; p += 256) {
        const float w = ivar[p];
        if (w > 0.f) { n += 1.0; sl += log((double)w); wm = fmax(wm, (double)w); }
    }
    for (int t = threadIdx.x; t < ktaps; t += 256) ps += fabs((double)psf[t]);
    r1[threadIdx.x] = n; r2[threadIdx.x] = sl; r3[threadIdx.x] = wm; r4[threadIdx.x] = ps;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            r1[threadIdx.x] += r1[threadIdx.x + o]; r2[threadIdx.x] += r2[threadIdx.x + o];
            r3[threadIdx.x] = fmax(r3[threadIdx.x], r3[threadIdx.x + o]); r4[threadIdx.x] += r4[threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { st[0] = r1[0]; st[1] = r2[0]; st[2] = r3[0] > 0.0 ? r3[0] : 1.0; st[3] = r4[0] > 0.0 ? r4[0] : 1.0; }
}

__global__ void pixsrc_final_kernel(const float* __restrict__ lens, const float* __restrict__ src_grid, const float* __restrict__ lam_reg,
                                    const float* __restrict__ ms_lambda, const double* __restrict__ out, const double* __restrict__ st,
                                    const double* __restrict__ s, double logdet_g, int B, int ns, int npix, float* __restrict__ logev,
                                    float* __restrict__ chi2, float* __restrict__ reg, float* __restrict__ s_mp, float* __restrict__ model,
                                    int32_t* __restrict__ flags) {
    const int b = blockIdx.x;
    if (b >= B) return;
    const float lam = lam_reg[b];
    bool valid = pixsrc_valid(lens + (size_t)b * GLAD_NLENS, lam, src_grid[(size_t)b * 3 + 2]);
    if (ms_lambda && !isfinite(ms_lambda[b])) valid = false;
    const bool notpd = out[(size_t)b * PX_OUT + 3] != 0.0;
    const bool ok = valid && !notpd;
    const float inf = __int_as_float(0x7f800000), nan = __int_as_float(0x7fc00000);
    if (threadIdx.x == 0) {
        const double c2 = out[(size_t)b * PX_OUT + 2], es = out[(size_t)b * PX_OUT + 1], ld = out[(size_t)b * PX_OUT + 0];
        const double ev = -0.5 * c2 - (double)lam * es - 0.5 * ld + 0.5 * ns * log((double)lam) + 0.5 * logdet_g -
                          0.5 * st[0] * 1.8378770664093454836 + 0.5 * st[1];
        if (logev) logev[b] = ok ? (float)ev : -inf;
        if (chi2) chi2[b] = ok ? (float)c2 : inf;
        if (reg) reg[b] = ok ? (float)es : nan;
        if (flags) flags[b] = (valid ? 0 : GLAD_FLAG_LENS_INVALID) | ((valid && notpd) ? GLAD_FLAG_PIXSRC_NOT_PD : 0);
    }
    if (s_mp)
        for (int i = threadIdx.x; i < ns; i += blockDim.x) s_mp[(size_t)b * ns + i] = ok ? (float)s[(size_t)b * ns + i] : nan;
    if (model && !ok)
        for (int i = threadIdx.x; i < npix; i += blockDim.x) model[(size_t)b * npix + i] = nan;
}

// ------------------------------------------------------------------------------------------------------------------
// launcher: one chunk of Bc vectors through the whole chain on c->stream.  Scratch layout (bytes): pixsrc_scratch_bytes.
// ------------------------------------------------------------------------------------------------------------------
static inline size_t px_align(size_t n) { return (n + 255) & ~(size_t)255; }

// ------------------------------------------------------------------------------------------------------------------
// lambda_hat of Eq. 43: F and D do not depend on lambda, only the factorisation does.  With (F + lambda g) s = D,
//   -chi2/2 - lambda E_S = -(d^T C^-1 d - D^T s)/2, so up to lambda-independent terms
//   ln P(lambda) = J(x) = y^T y / 2 - ln det(F + e^x g) / 2 + N_s x / 2,  x = ln lambda, L y = D the forward substitution.
// Per vector: PX_GOLD golden-section steps on [ln lam_lo, ln lam_hi] (one Cholesky each), then the vertex of the parabola through
// the last bracket (a, better interior point, b); lambda_hat is rounded to the float32 the evidence entry takes.
// ------------------------------------------------------------------------------------------------------------------
#define PX_GOLD 18
#define PX_PHI 0.6180339887498949
struct PxSearch { double a, b, x1, x2, f1, f2, fa, fb; int which, pad; };   // which: the interior point (1 or 2) whose value is being computed

// A = F + lambda g on the lower triangle
__global__ void __launch_bounds__(256) pixsrc_shift_kernel(const double* __restrict__ F, const double* __restrict__ lam, int ns, int nsx,
                                                           int nsy, double* __restrict__ A) {
    const int b = blockIdx.y;
    const size_t e = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (e >= (size_t)ns * ns) return;
    const int i = (int)(e / ns), j = (int)(e - (size_t)i * ns);
    if (j > i) return;
    A[(size_t)b * ns * ns + e] = F[(size_t)b * ns * ns + e] + lam[b] * px_curv(i, j, nsx, nsy);
}

__device__ __forceinline__ double px_objective(const double* __restrict__ o, int ns, double x) {
    if (o[3] != 0.0 || !isfinite(o[0]) || !isfinite(o[4])) return -__longlong_as_double(0x7ff0000000000000LL);   // not positive definite
    return 0.5 * o[4] - 0.5 * o[0] + 0.5 * ns * x;
}

// step -2: set up the bracket and ask for J(a); -1: store J(a), ask J(b); 0: store J(b), ask J(x1); 1: store J(x1), ask J(x2);
// 2..: one golden-section step per call; last: parabola vertex -> lam_hat
__global__ void pixsrc_search_kernel(PxSearch* __restrict__ st, const double* __restrict__ out, int B, int ns, double xlo, double xhi,
                                     int step, int last, double* __restrict__ lam_cur, float* __restrict__ lam_hat) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    PxSearch s = st[b];
    const double* o = out + (size_t)b * PX_OUT;
    double ask;
    if (step == -2) {
        s.a = xlo; s.b = xhi;
        s.x1 = s.b - PX_PHI * (s.b - s.a); s.x2 = s.a + PX_PHI * (s.b - s.a);
        ask = s.a;
    } else if (step == -1) { s.fa = px_objective(o, ns, s.a); ask = s.b; }
    else if (step == 0) { s.fb = px_objective(o, ns, s.b); ask = s.x1; }
    else if (step == 1) { s.f1 = px_objective(o, ns, s.x1); ask = s.x2; s.which = 2; }
    else {
        if (s.which == 1) s.f1 = px_objective(o, ns, s.x1);
        else s.f2 = px_objective(o, ns, s.x2);
        if (!last) {
            if (s.f1 > s.f2) { s.b = s.x2; s.fb = s.f2; s.x2 = s.x1; s.f2 = s.f1; s.x1 = s.b - PX_PHI * (s.b - s.a); ask = s.x1; s.which = 1; }
            else { s.a = s.x1; s.fa = s.f1; s.x1 = s.x2; s.f1 = s.f2; s.x2 = s.a + PX_PHI * (s.b - s.a); ask = s.x2; s.which = 2; }
        } else {
            // vertex of the parabola through (a, fa), (m, fm), (b, fb), m = the better interior point; kept inside the bracket
            const double m = s.f1 > s.f2 ? s.x1 : s.x2, fm = s.f1 > s.f2 ? s.f1 : s.f2;
            double x = m;
            const double d1 = (m - s.a) * (fm - s.fb), d2 = (m - s.b) * (fm - s.fa);
            const double den = d1 - d2;
            if (isfinite(s.fa) && isfinite(s.fb) && isfinite(fm) && den != 0.0) {
                const double v = m - 0.5 * ((m - s.a) * d1 - (m - s.b) * d2) / den;
                if (v > s.a && v < s.b) x = v;
            }
            lam_hat[b] = (float)exp(x);
            ask = x;
        }
    }
    lam_cur[b] = last ? (double)lam_hat[b] : exp(ask);
    st[b] = s;
}

static inline size_t px_ntiles(int ns) { const size_t nt = (ns + 127) / 128; return nt * (nt + 1) / 2; }   // output tiles of the contraction
size_t pixsrc_scratch_bytes(int npix, int ns, int Bc, bool search) {
    return px_align(sizeof(int) * (size_t)Bc * npix) + px_align(sizeof(float2) * (size_t)Bc * npix) + px_align(sizeof(int2) * (size_t)Bc * npix) +
           px_align(sizeof(float) * (size_t)Bc * npix * ns) + (search ? 2 : 1) * px_align(sizeof(double) * (size_t)Bc * ns * ns) +
           2 * px_align(sizeof(double) * (size_t)Bc * ns) + px_align(sizeof(double) * (size_t)Bc * PX_OUT) + px_align(sizeof(double) * 4) +
           (search ? px_align(sizeof(PxSearch) * (size_t)Bc) + px_align(sizeof(double) * (size_t)Bc) + px_align(sizeof(float) * (size_t)Bc) : 0) +
           px_align(sizeof(unsigned short) * (size_t)Bc * px_ntiles(ns) * npix) + px_align(pixsrc_factor_scratch_bytes(Bc));
}

// d_lam != NULL: the evidence at the given lambda; d_lam == NULL: search lambda_hat on [lam_lo, lam_hi] first, write it to d_lam_hat
cudaError_t launch_pixsrc_chunk(glad_ctx* c, void* scratch, const float* d_lens, const float* d_src_grid, const float* d_lam,
                                const float* d_ms_lambda, int nsx, int nsy, int Bc, double logdet_g, float* d_logev, float* d_chi2,
                                float* d_reg, float* d_s_mp, float* d_model, int32_t* d_flags, double lam_lo, double lam_hi,
                                float* d_lam_hat) {
    const bool search = d_lam == nullptr;
    const int nx = c->grid.nx, ny = c->grid.ny, npix = nx * ny, ns = nsx * nsy;
    cudaStream_t st = c->stream;
    char* q = (char*)scratch;
    int* idx = (int*)q;            q += px_align(sizeof(int) * (size_t)Bc * npix);
    float2* wgt = (float2*)q;      q += px_align(sizeof(float2) * (size_t)Bc * npix);
    int2* rng = (int2*)q;          q += px_align(sizeof(int2) * (size_t)Bc * npix);
    float* f = (float*)q;          q += px_align(sizeof(float) * (size_t)Bc * npix * ns);
    double* A = (double*)q;        q += px_align(sizeof(double) * (size_t)Bc * ns * ns);
    double* D = (double*)q;        q += px_align(sizeof(double) * (size_t)Bc * ns);
    double* s = (double*)q;        q += px_align(sizeof(double) * (size_t)Bc * ns);
    double* out = (double*)q;      q += px_align(sizeof(double) * (size_t)Bc * PX_OUT);
    double* stat = (double*)q;     q += px_align(sizeof(double) * 4);
    double* Fm = nullptr; PxSearch* sst = nullptr; double* lam_cur = nullptr; float* lam_f = nullptr;
    if (search) {
        Fm = (double*)q;           q += px_align(sizeof(double) * (size_t)Bc * ns * ns);
        sst = (PxSearch*)q;        q += px_align(sizeof(PxSearch) * (size_t)Bc);
        lam_cur = (double*)q;      q += px_align(sizeof(double) * (size_t)Bc);
        lam_f = (float*)q;         q += px_align(sizeof(float) * (size_t)Bc);
    }
    unsigned short* rowlist = (unsigned short*)q;   q += px_align(sizeof(unsigned short) * (size_t)Bc * px_ntiles(ns) * npix);
    double* Winv = (double*)q;
    cudaError_t e;
    if ((e = cudaMemsetAsync(out, 0, sizeof(double) * (size_t)Bc * PX_OUT, st)) != cudaSuccess) return e;

    const int rows_per_cta = 64;
    const size_t sm_blur = sizeof(float) * (size_t)PX_BLUR_WARPS * ns;
    const size_t sm_chol = sizeof(double) * ((size_t)ns + 8 * 32 + PX_NB * (PX_NB + 1));
    if (sm_blur > 227 * 1024 || sm_chol > 227 * 1024) return cudaErrorInvalidConfiguration;
    if ((e = smem_optin(c, pixsrc_blur_kernel)) != cudaSuccess) return e;
    if ((e = smem_optin(c, pixsrc_solve_kernel)) != cudaSuccess) return e;
    pixsrc_static_kernel<<<1, 256, 0, st>>>(c->d_ivar, npix, c->d_psf, c->kpsf * c->kpsf, stat);
    c->launches++;
    {
        ProfScope ps(c, GK_PIX_MAP);
        pixsrc_map_kernel<<<dim3((npix + PX_MAP_THREADS - 1) / PX_MAP_THREADS, Bc), PX_MAP_THREADS, 0, st>>>(
            d_lens, d_src_grid, d_lam, d_ms_lambda, c->ms_rc, c->ms_rt, c->grid, nsx, nsy, idx, wgt);
    }
    {
        ProfScope ps(c, GK_PIX_BLUR);
        pixsrc_blur_kernel<<<dim3((npix + rows_per_cta - 1) / rows_per_cta, Bc), 32 * PX_BLUR_WARPS, sm_blur, st>>>(
            idx, wgt, c->d_psf, c->kpsf, nx, ny, nsx, ns, rows_per_cta, f, rng, stat);
    }
    {
        // F (+ lambda g) and D in one pass over f on the tensor cores (pixsrc_syrk_tc.cu)
        ProfScope ps(c, GK_PIX_SYRK);
        if ((e = launch_pixsrc_syrk_tc(c, st, f, rng, d_lam, npix, ns, nsx, nsy, Bc, stat, rowlist, search ? Fm : A, D)) != cudaSuccess) return e;
    }
    const float* lam_use = d_lam;
    if (search) {
        // Eq. 43: PX_GOLD golden-section steps, each = A <- F + lambda g, Cholesky + forward substitution, bracket update; all on
        // the stream, no host round trip
        const dim3 gs((unsigned)(((size_t)ns * ns + 255) / 256), Bc);
        const int last_step = 2 + PX_GOLD;
        for (int step = -2; step <= last_step; ++step) {
            pixsrc_search_kernel<<<(Bc + 127) / 128, 128, 0, st>>>(sst, out, Bc, ns, log(lam_lo), log(lam_hi), step, step == last_step, lam_cur, lam_f);
            c->launches++;
            pixsrc_shift_kernel<<<gs, 256, 0, st>>>(Fm, lam_cur, ns, nsx, nsy, A);
            c->launches++;
            if (step == last_step) break;
            ProfScope ps(c, GK_PIX_CHOL);
            if ((e = launch_pixsrc_factor(c, st, A, ns, Bc, out, Winv)) != cudaSuccess) return e;
            pixsrc_solve_kernel<<<Bc, PX_CHOL_THREADS, sm_chol, st>>>(A, D, ns, nsx, nsy, s, out, 1);
        }
        lam_use = lam_f;
        if (d_lam_hat && (e = cudaMemcpyAsync(d_lam_hat, lam_f, sizeof(float) * Bc, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return e;
    }
    {
        ProfScope ps(c, GK_PIX_CHOL);
        if ((e = launch_pixsrc_factor(c, st, A, ns, Bc, out, Winv)) != cudaSuccess) return e;
        pixsrc_solve_kernel<<<Bc, PX_CHOL_THREADS, sm_chol, st>>>(A, D, ns, nsx, nsy, s, out, 0);
    }
    {
        ProfScope ps(c, GK_PIX_MODEL);
        pixsrc_model_kernel<<<dim3((npix + 63) / 64, Bc), 256, sizeof(double) * ns, st>>>(f, s, c->d_ivar, c->d_data, npix, ns, d_model,
                                                                                          (long)npix, out, rng);
    }
    pixsrc_final_kernel<<<Bc, 128, 0, st>>>(d_lens, d_src_grid, lam_use, d_ms_lambda, out, stat, s, logdet_g, Bc, ns, npix, d_logev, d_chi2,
                                            d_reg, d_s_mp, d_model, d_flags);
    c->launches++;
    return cudaGetLastError();
}
