// JAM_sph, the dynamics the paper runs (Eq. 17-20; Eq. 26; fixed mesh P:358-362).
// Axisymmetric Jeans model with a spherically-aligned velocity ellipsoid on MGE tracer and mass.  DESIGN.md R-SPH1..6 state the
// solution (characteristics of Eq. 17-18: sin th' = sin th (r/r')^(1-beta)) and every choice the paper leaves open.
//
//   jam_sph_prep_kernel   per vector, fp64 -> fp32: deprojected luminous Gaussians, anisotropy groups, and the potential table
//                         over (mass Gaussian j, node u_m): {p, d, w0, w1, w2} with
//                           p = log2e u^2 / (2 s_j^2 g), d = -p e_j u^2, g = 1 - e_j u^2   (exponent = -(r'^2 p + r'^2 s'^2 d))
//                           w0 = w_m C_j u^2 / (s_j^2 g^(3/2)),  w1 = w0 e_j u^4 / (s_j^2 g),  w2 = w0 e_j u^2.
//   jam_sph_intr_kernel   THE hot loop (the paper's "main computational bottleneck"): for every polar grid point and
//                         radial node, sum the table: S0 = sum w0 E, S1 = sum w1 E, E = 2^-(c2 p + c1 d).  One thread per
//                         (point, node) pair, the table broadcast from shared memory.  Psi = nu x (potential term) is a PRODUCT
//                         of a sum over luminous Gaussians and a sum over (j, u) whenever the Gaussians share beta (the paper
//                         samples one beta_ani): (n_l + n_m n_u) exponentials per pair instead of n_l n_m n_u; Gaussians
//                         with different beta_k are handled group by group (each group has its own characteristics).
//   jam_sph_los_kernel    Eq. 26: per folded sky pixel, the LOS integral of nu v_z'^2 with the three moment ratios interpolated on
//                         the polar grid; writes the Sigma v^2 map that jam_post_kernel (rows a7-a8) bins.
#include <math.h>

#include "glad_internal.h"

#define SPH_LOG2E 1.4426950408889634
#define SPH_G 0.004301               // (km/s)^2 pc / Msun (R-D1)
#define SPH_SIGMA_BH 0.01            // arcsec (R-D3)
#define SPH_RCUT_SIGMAS 6.0          // R-SPH1
#define SPH_HDR 8
enum SphHdr { SH_RCUT = 0, SH_NGROUPS, SH_NM, SH_SINI, SH_COSI };
#define SPH_LUM 8                    // per luminous Gaussian: nu_n, pk, dk, ek, beta, group, -, -
enum SphLum { SL_NU = 0, SL_PK, SL_DK, SL_EK, SL_BETA, SL_GROUP };

// table layout (floats): header | nl x SPH_LUM | group betas (nl, padded to a multiple of 4) | nmx*nu float4 entries | nmx*nu w2;
// every part starts on a 16-byte boundary and so does every vector's table
static inline __host__ __device__ size_t sph_groups_floats(int nl) { return (size_t)((nl + 3) & ~3); }
static inline __host__ __device__ size_t sph_table_floats(int nl, int nmx, int nu) {
    return ((size_t)SPH_HDR + (size_t)SPH_LUM * nl + sph_groups_floats(nl) + (size_t)nmx * nu * 5 + 3) & ~(size_t)3;
}

__device__ __forceinline__ float sph_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sph_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__global__ void __launch_bounds__(128) jam_sph_prep_kernel(const float* __restrict__ dyn, const float* __restrict__ lum, int nl,
                                                          long lum_stride, const float* __restrict__ mass, int nm,
                                                          long mass_stride, const float* __restrict__ beta, int per_gaussian,
                                                          const float* __restrict__ un, const float* __restrict__ uw, int nu,
                                                          float* __restrict__ tab) {
    const int b = blockIdx.x, tid = threadIdx.x, nmx = nm + 1;
    float* T = tab + (size_t)b * sph_table_floats(nl, nmx, nu);
    float* TL = T + SPH_HDR;
    float* TG = TL + SPH_LUM * nl;            // beta of each anisotropy group
    float* TE = TG + sph_groups_floats(nl);   // entries: [nmx*nu] x {p, d, w0, w1} then [nmx*nu] x w2
    float* TW2 = TE + (size_t)4 * nmx * nu;
    __shared__ double s_max[128];
    const double PI = 3.14159265358979323846;
    const double inc = dyn[b * GLAD_NDYN + 0], Dd = dyn[b * GLAD_NDYN + 1];
    const double Mbh = dyn[b * GLAD_NDYN + 2], ups = dyn[b * GLAD_NDYN + 3];
    const double ci = cos(inc), si = sin(inc), ci2 = ci * ci;
    const double pc = Dd * PI / 0.648;
    const float* lt = lum + (size_t)b * lum_stride;
    const float* mt = mass + (size_t)b * mass_stride;
    const bool has_bh = Mbh > 0.0;
    double smax = 0.0;
    for (int k = tid; k < nl; k += blockDim.x) {
        double I0 = lt[3 * k], sg = lt[3 * k + 1], qp = lt[3 * k + 2];
        double bz = per_gaussian ? beta[(size_t)b * nl + k] : beta[b];
        double d = qp * qp - ci2;
        if (!(d > 0.0) || !(sg > 0.0) || !(qp > 0.0) || !(si > 0.0)) { d = 1.0; sg = 1.0; qp = 1.0; }   // invalid: flagged by jam_prep
        double q = sqrt(d) / si, q2 = q * q, s2 = sg * sg;
        double a = SPH_LOG2E / (2.0 * s2), bq = 1.0 / q2;
        TL[SPH_LUM * k + SL_NU] = (float)(I0 * qp / (q * sg * sqrt(2.0 * PI)));     // Eq. 23, per pc^2 per arcsec
        TL[SPH_LUM * k + SL_PK] = (float)(a * bq);
        TL[SPH_LUM * k + SL_DK] = (float)(a * (1.0 - bq));
        TL[SPH_LUM * k + SL_EK] = (float)((1.0 - q2) / (s2 * q2));
        TL[SPH_LUM * k + SL_BETA] = (float)bz;
        if (sg > smax) smax = sg;
    }
    s_max[tid] = smax;
    __syncthreads();
    if (tid == 0) {
        for (int i = 1; i < (int)blockDim.x; ++i) if (s_max[i] > smax) smax = s_max[i];
        // anisotropy groups: Gaussians with bitwise equal beta share their characteristics
        int ng = 0;
        for (int k = 0; k < nl; ++k) {
            const float bk = TL[SPH_LUM * k + SL_BETA];
            int g = -1;
            for (int h = 0; h < ng; ++h) if (TG[h] == bk) { g = h; break; }
            if (g < 0) { g = ng; TG[ng++] = bk; }
            TL[SPH_LUM * k + SL_GROUP] = __int_as_float(g);
        }
        T[SH_RCUT] = (float)(SPH_RCUT_SIGMAS * smax);
        T[SH_NGROUPS] = __int_as_float(ng);
        T[SH_NM] = __int_as_float(has_bh ? nmx : nm);
        T[SH_SINI] = (float)si;
        T[SH_COSI] = (float)ci;
    }
    const int ne = nmx * nu;
    for (int e = tid; e < ne; e += blockDim.x) {
        const int j = e / nu, m = e - j * nu;
        double sg, q2, Cj;
        if (j < nm) {
            double S0 = ups * (double)mt[3 * j], qp = mt[3 * j + 2];
            sg = mt[3 * j + 1];
            double d = qp * qp - ci2;
            if (!(d > 0.0) || !(sg > 0.0) || !(qp > 0.0) || !(si > 0.0)) { d = 1.0; sg = 1.0; qp = 1.0; S0 = 0.0; }
            q2 = d / (si * si);
            // C_j = sqrt(2/pi) G M_j / sigma_j[pc], M_j = 2 pi Sigma_0j (sigma_j pc)^2 q'_j, lengths otherwise in arcsec
            Cj = sqrt(2.0 / PI) * 2.0 * PI * SPH_G * pc * S0 * sg * qp;
        } else {
            sg = SPH_SIGMA_BH; q2 = 1.0;
            Cj = has_bh ? sqrt(2.0 / PI) * SPH_G * Mbh / (pc * sg) : 0.0;
        }
        const double ej = 1.0 - q2, u = un[m], u2 = u * u, g = 1.0 - ej * u2, s2 = sg * sg;
        const double p = SPH_LOG2E * u2 / (2.0 * s2 * g);
        const double w0 = (double)uw[m] * Cj * u2 / (s2 * g * sqrt(g));
        TE[4 * e + 0] = (float)p;
        TE[4 * e + 1] = (float)(-p * ej * u2);
        TE[4 * e + 2] = (float)w0;
        TE[4 * e + 3] = (float)(w0 * ej * u2 * u2 / (s2 * g));
        TW2[e] = (float)(w0 * ej * u2);
    }
}

struct SphIntrArgs {
    const float* tab; size_t tabsz; const float* jtab; int jtabsz;
    int nl, nmx, nu;
    const float* rgrid; int nr; const float* thgrid; int nth;
    const float* tau; const float* wtau; int nt;
    int ppc;            // polar points per CTA
    int nchunk;         // CTAs per vector
    float* ratios;      // [B,3,nr,nth]
};

// CTA = (vector, chunk of polar points).  Shared memory: the vector's potential table (nm*nu float4 + w2), its luminous
// Gaussians, and three partial sums per (point, node) pair of the chunk.
__global__ void __launch_bounds__(256) jam_sph_intr_kernel(SphIntrArgs a) {
    extern __shared__ __align__(16) float sm[];
    const int b = blockIdx.x / a.nchunk, chunk = blockIdx.x - b * a.nchunk;
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const float* T = a.tab + (size_t)b * a.tabsz;
    const int npol = a.nr * a.nth;
    float* out = a.ratios + (size_t)b * 3 * npol;
    const int p0 = chunk * a.ppc, p1 = min(p0 + a.ppc, npol);
    const float qnan = __int_as_float(0x7fc00000);
    if (__float_as_int(a.jtab[(size_t)b * a.jtabsz + JH_VALID]) == 0) {
        for (int i = p0 + tid; i < p1; i += nthr) { out[i] = qnan; out[npol + i] = qnan; out[2 * npol + i] = qnan; }
        return;
    }
    const int nl = a.nl, nt = a.nt;
    const int nm = __float_as_int(T[SH_NM]), ng = __float_as_int(T[SH_NGROUPS]);
    const int ne = nm * a.nu;                               // a vector without black hole skips the last Gaussian's entries
    float4* s_e = reinterpret_cast<float4*>(sm);            // [ne]
    float* s_w2 = sm + 4 * (size_t)a.nmx * a.nu;            // [ne]
    float* s_l = s_w2 + (size_t)a.nmx * a.nu;               // [nl][SPH_LUM]
    float* s_g = s_l + SPH_LUM * nl;                        // [nl] group betas (padded)
    float* s_part = s_g + sph_groups_floats(nl);            // [ppc*nt][3]
    float* s_pt = s_part + 3 * (size_t)a.ppc * nt;          // [ppc][2]: nu, P
    {
        const size_t off = SPH_HDR + (size_t)SPH_LUM * nl + sph_groups_floats(nl);
        const float4* ge = reinterpret_cast<const float4*>(T + off);
        for (int i = tid; i < ne; i += nthr) s_e[i] = ge[i];
        const float* gw = T + off + 4 * (size_t)a.nmx * a.nu;
        for (int i = tid; i < ne; i += nthr) s_w2[i] = gw[i];
        for (int i = tid; i < SPH_LUM * nl + nl; i += nthr) s_l[i] = T[SPH_HDR + i];
    }
    const int npairs = (p1 - p0) * nt;
    for (int i = tid; i < 3 * npairs; i += nthr) s_part[i] = 0.f;
    __syncthreads();
    const float rcut = T[SH_RCUT];

    for (int g = 0; g < ng; ++g) {
        const float betag = s_g[g], omb = 1.f - betag;
        for (int pr = tid; pr < npairs; pr += nthr) {
            const int pl = pr / nt, n = pr - pl * nt, pt = p0 + pl;
            const int ia = pt / a.nth, it = pt - ia * a.nth;
            const float r = a.rgrid[ia];
            if (!(rcut > r)) continue;
            const float sth = sinf(a.thgrid[it]);
            const float s2 = sth * sth;
            const float W2 = sph_lg2(rcut / r);               // log2(r_cut / r)
            const float x = W2 * a.tau[n];                    // log2(r'/r)
            const float rp = r * sph_ex2(x);
            const float c2 = rp * rp;
            const float c1 = c2 * s2 * sph_ex2(-2.f * omb * x);   // r'^2 sin^2 theta' on the characteristic
            float A0 = 0.f, A1 = 0.f;                         // sum_k nu_k, sum_k nu_k e_k/(s_k^2 q_k^2) over the group
            for (int k = 0; k < nl; ++k) {
                const float* L = s_l + SPH_LUM * k;
                if (__float_as_int(L[SL_GROUP]) != g) continue;
                const float nuk = L[SL_NU] * sph_ex2(-fmaf(c2, L[SL_PK], c1 * L[SL_DK]));
                A0 += nuk;
                A1 = fmaf(nuk, L[SL_EK], A1);
            }
            float S0a = 0.f, S0b = 0.f, S1a = 0.f, S1b = 0.f;
            int e = 0;
            for (; e + 1 < ne; e += 2) {                      // two independent chains: the MUFU latency is covered
                const float4 t0 = s_e[e], t1 = s_e[e + 1];
                const float E0 = sph_ex2(-fmaf(c2, t0.x, c1 * t0.y));
                const float E1 = sph_ex2(-fmaf(c2, t1.x, c1 * t1.y));
                S0a = fmaf(t0.z, E0, S0a); S1a = fmaf(t0.w, E0, S1a);
                S0b = fmaf(t1.z, E1, S0b); S1b = fmaf(t1.w, E1, S1b);
            }
            if (e < ne) {
                const float4 t0 = s_e[e];
                const float E0 = sph_ex2(-fmaf(c2, t0.x, c1 * t0.y));
                S0a = fmaf(t0.z, E0, S0a); S1a = fmaf(t0.w, E0, S1a);
            }
            const float S0 = S0a + S0b, S1 = S1a + S1b;
            // dr'/r' = ln(r_cut/r) dtau;  (r'/r)^(2 beta)
            const float jac = W2 * 0.6931471805599453f * a.wtau[n] * sph_ex2(2.f * betag * x) * c2;
            const float F = jac * A0 * S0;
            const float Gd = jac * c1 * fmaf(A1, S0, A0 * S1);
            float* o = s_part + 3 * pr;
            o[0] += F;
            o[1] = fmaf(omb, F, o[1]);
            o[2] = fmaf(omb, F + Gd, o[2]);
        }
    }
    // the point itself: nu and nu tan(theta) dPhi/dtheta = -nu r^2 s^2 sum w2 E: a warp per point
    for (int pl = warp; pl < p1 - p0; pl += nthr >> 5) {
        const int pt = p0 + pl, ia = pt / a.nth, it = pt - ia * a.nth;
        const float r = a.rgrid[ia], sth = sinf(a.thgrid[it]), s2 = sth * sth;
        const float c2 = r * r, c1 = c2 * s2;
        float acc = 0.f, nu = 0.f;
        for (int e = lane; e < ne; e += 32) {
            const float4 t0 = s_e[e];
            acc = fmaf(s_w2[e], sph_ex2(-fmaf(c2, t0.x, c1 * t0.y)), acc);
        }
        for (int k = lane; k < nl; k += 32) {
            const float* L = s_l + SPH_LUM * k;
            nu += L[SL_NU] * sph_ex2(-fmaf(c2, L[SL_PK], c1 * L[SL_DK]));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc += __shfl_xor_sync(0xffffffffu, acc, o);
            nu += __shfl_xor_sync(0xffffffffu, nu, o);
        }
        if (lane == 0) { s_pt[2 * pl] = nu; s_pt[2 * pl + 1] = -nu * c1 * acc; }
    }
    __syncthreads();
    // nodes summed in order (deterministic), then the ratios v_r^2, v_th^2, v_phi^2 = (nu v^2) / nu
    for (int pl = tid; pl < p1 - p0; pl += nthr) {
        float Tr = 0.f, Tt = 0.f, Tp = 0.f;
        for (int n = 0; n < nt; ++n) {
            const float* o = s_part + 3 * (pl * nt + n);
            Tr += o[0]; Tt += o[1]; Tp += o[2];
        }
        const float nu = s_pt[2 * pl];
        Tp += s_pt[2 * pl + 1];
        const float inv = nu > 0.f ? 1.f / nu : 0.f;
        out[p0 + pl] = Tr * inv;
        out[npol + p0 + pl] = Tt * inv;
        out[2 * npol + p0 + pl] = Tp * inv;
    }
}

struct SphLosArgs {
    const float* tab; size_t tabsz; const float* jtab; int jtabsz;
    int nl;
    const float* rgrid; int nr; const float* thgrid; int nth;
    const float* zeta; const float* wz; int nz;
    const float* xf; const float* yf; int nxf, nyf;
    const float* ratios;    // [B,3,nr,nth]
    float* partial;         // [B,nyf*nxf]
};

// Eq. 26: thread per folded sky pixel, loop over the LOS nodes (R-SPH3..5)
__global__ void __launch_bounds__(128) jam_sph_los_kernel(SphLosArgs a) {
    extern __shared__ __align__(16) float sm[];
    const int b = blockIdx.y, tid = threadIdx.x, nthr = blockDim.x;
    if (__float_as_int(a.jtab[(size_t)b * a.jtabsz + JH_VALID]) == 0) return;     // jam_post_kernel never reads this vector's map
    const float* T = a.tab + (size_t)b * a.tabsz;
    const int npol = a.nr * a.nth, nl = a.nl;
    float* s_rat = sm;                        // [3][npol]
    float* s_lr = s_rat + 3 * npol;           // [nr] ln r_a
    float* s_th = s_lr + a.nr;                // [nth]
    float* s_l = s_th + a.nth;                // [nl][3]: nu_n, pk, dk
    float* s_z = s_l + 3 * nl;                // [nz][2]
    for (int i = tid; i < 3 * npol; i += nthr) s_rat[i] = a.ratios[(size_t)b * 3 * npol + i];
    for (int i = tid; i < a.nr; i += nthr) s_lr[i] = logf(a.rgrid[i]);
    for (int i = tid; i < a.nth; i += nthr) s_th[i] = a.thgrid[i];
    for (int i = tid; i < nl; i += nthr) {
        const float* L = T + SPH_HDR + SPH_LUM * i;
        s_l[3 * i] = L[SL_NU]; s_l[3 * i + 1] = L[SL_PK]; s_l[3 * i + 2] = L[SL_DK];
    }
    for (int i = tid; i < a.nz; i += nthr) { s_z[2 * i] = a.zeta[i]; s_z[2 * i + 1] = a.wz[i]; }
    __syncthreads();
    const int npf = a.nxf * a.nyf, i = blockIdx.x * nthr + tid;
    if (i >= npf) return;
    const int fy = i / a.nxf, fx = i - fy * a.nxf;
    const float xp = a.xf[fx], yp = a.yf[fy];
    const float si = T[SH_SINI], ci = T[SH_COSI], rcut = T[SH_RCUT];
    const float rho = sqrtf(fmaf(xp, xp, yp * yp));
    const float rho0 = fmaxf(rho, a.rgrid[0]);
    const float aa = asinhf(rcut / rho0);
    const int nr = a.nr, nth = a.nth;
    float total = 0.f;
    for (int n = 0; n < a.nz; ++n) {
        const float ez = __expf(aa * s_z[2 * n]), iez = 1.f / ez;
        const float zp = 0.5f * rho0 * (ez - iez);
        const float dz = 0.5f * rho0 * aa * (ez + iez) * s_z[2 * n + 1];
        const float y = fmaf(zp, si, -yp * ci), z = fmaf(yp, si, zp * ci);
        const float R2 = fmaf(xp, xp, y * y), r2 = fmaf(z, z, R2);
        if (!(r2 > 0.f)) continue;
        const float rinv = rsqrtf(r2), R = sqrtf(R2);
        const float ct = z * rinv, st = R * rinv, c1 = R2;            // r^2 sin^2 theta = R^2
        float nu = 0.f;
        for (int k = 0; k < nl; ++k) nu += s_l[3 * k] * sph_ex2(-fmaf(r2, s_l[3 * k + 1], c1 * s_l[3 * k + 2]));
        const float lr = 0.5f * __logf(r2);
        const float t = acosf(fminf(fabsf(ct), 1.f));
        int ia = 0, ib = 0;
        float fa = 0.f, fb = 0.f;
        if (nr > 1) {
            if (lr <= s_lr[0]) { ia = 0; fa = 0.f; }
            else if (lr >= s_lr[nr - 1]) { ia = nr - 2; fa = 1.f; }
            else { while (ia < nr - 2 && lr >= s_lr[ia + 1]) ++ia; fa = (lr - s_lr[ia]) / (s_lr[ia + 1] - s_lr[ia]); }
        }
        if (nth > 1) {
            if (t <= s_th[0]) { ib = 0; fb = 0.f; }
            else if (t >= s_th[nth - 1]) { ib = nth - 2; fb = 1.f; }
            else { while (ib < nth - 2 && t >= s_th[ib + 1]) ++ib; fb = (t - s_th[ib]) / (s_th[ib + 1] - s_th[ib]); }
        }
        const int ia1 = nr > 1 ? ia + 1 : ia, ib1 = nth > 1 ? ib + 1 : ib;
        const float w00 = (1.f - fa) * (1.f - fb), w01 = (1.f - fa) * fb, w10 = fa * (1.f - fb), w11 = fa * fb;
        const int i00 = ia * nth + ib, i01 = ia * nth + ib1, i10 = ia1 * nth + ib, i11 = ia1 * nth + ib1;
        const float vr2 = w00 * s_rat[i00] + w01 * s_rat[i01] + w10 * s_rat[i10] + w11 * s_rat[i11];
        const float vt2 = w00 * s_rat[npol + i00] + w01 * s_rat[npol + i01] + w10 * s_rat[npol + i10] + w11 * s_rat[npol + i11];
        const float vp2 = w00 * s_rat[2 * npol + i00] + w01 * s_rat[2 * npol + i01] + w10 * s_rat[2 * npol + i10] + w11 * s_rat[2 * npol + i11];
        const float Rinv = R > 0.f ? 1.f / R : 0.f;
        const float cph = R > 0.f ? xp * Rinv : 1.f, sph = y * Rinv;
        const float pr = zp * rinv, pt = fmaf(ct * sph, si, -st * ci), pp = cph * si;
        total = fmaf(dz * nu, fmaf(vr2 * pr, pr, fmaf(vt2 * pt, pt, vp2 * pp * pp)), total);
    }
    a.partial[(size_t)b * npf + i] = total;
}

size_t jam_sph_table_floats(int nl, int nmx, int nu) { return sph_table_floats(nl, nmx, nu); }

// shared memory of the hot kernel for `ppc` polar points per CTA
static size_t sph_intr_smem(int nl, int nmx, int nu, int nt, int ppc) {
    return sizeof(float) * (5 * (size_t)nmx * nu + (size_t)SPH_LUM * nl + sph_groups_floats(nl) + 3 * (size_t)ppc * nt + 2 * (size_t)ppc);
}

bool jam_sph_supported(const glad_ctx* c, int nl, int nmx) {
    return sph_intr_smem(nl, nmx, c->sph_nu, c->sph_nt, 1) <= (size_t)glad_smem_dynamic_max(c);
}

cudaError_t launch_jam_sph(glad_ctx* c, const float* d_dyn, int B, const float* d_lum, int nl, long lum_stride,
                           const float* d_mass, int nm, long mass_stride, const float* d_beta, int per_gaussian,
                           float* d_ratios) {
    const int nmx = nm + 1, nu = c->sph_nu, nt = c->sph_nt, npol = c->sph_nr * c->sph_nth;
    const size_t tabsz = sph_table_floats(nl, nmx, nu);
    {
        ProfScope ps(c, GK_JAM_PREP);
        jam_sph_prep_kernel<<<B, 128, 0, c->stream>>>(d_dyn, d_lum, nl, lum_stride, d_mass, nm, mass_stride, d_beta, per_gaussian,
                                                     c->d_sph_un, c->d_sph_uw, nu, c->d_sph_tab);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    // points per CTA: about 2048 (point, node) pairs each, and enough CTAs to fill the device when the batch is small
    int ppc = (2048 + nt - 1) / nt;
    while (ppc > 1 && (long)B * ((npol + ppc - 1) / ppc) < 2L * c->sm_count) --ppc;
    while (ppc > 1 && sph_intr_smem(nl, nmx, nu, nt, ppc) > (size_t)glad_smem_dynamic_max(c)) --ppc;
    const size_t smem = sph_intr_smem(nl, nmx, nu, nt, ppc);
    if (smem > (size_t)glad_smem_dynamic_max(c)) return cudaErrorInvalidConfiguration;
    SphIntrArgs a;
    a.tab = c->d_sph_tab; a.tabsz = tabsz; a.jtab = c->d_jam_tab; a.jtabsz = jam_table_floats(nl, nmx);
    a.nl = nl; a.nmx = nmx; a.nu = nu;
    a.rgrid = c->d_sph_r; a.nr = c->sph_nr; a.thgrid = c->d_sph_th; a.nth = c->sph_nth;
    a.tau = c->d_sph_tau; a.wtau = c->d_sph_wtau; a.nt = nt;
    a.ppc = ppc; a.nchunk = (npol + ppc - 1) / ppc; a.ratios = d_ratios;
    cudaError_t e = smem_optin(c, jam_sph_intr_kernel);
    if (e != cudaSuccess) return e;
    {
        ProfScope ps(c, GK_JAM_SPH);
        jam_sph_intr_kernel<<<B * a.nchunk, 256, smem, c->stream>>>(a);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    SphLosArgs l;
    l.tab = c->d_sph_tab; l.tabsz = tabsz; l.jtab = a.jtab; l.jtabsz = a.jtabsz; l.nl = nl;
    l.rgrid = a.rgrid; l.nr = a.nr; l.thgrid = a.thgrid; l.nth = a.nth;
    l.zeta = c->d_sph_zeta; l.wz = c->d_sph_wz; l.nz = c->sph_nz;
    l.xf = c->d_xf; l.yf = c->d_yf; l.nxf = c->nxf; l.nyf = c->nyf;
    l.ratios = d_ratios; l.partial = c->d_partial;
    const size_t smem2 = sizeof(float) * (3 * (size_t)npol + a.nr + a.nth + 3 * (size_t)nl + 2 * (size_t)c->sph_nz);
    if (smem2 > (size_t)glad_smem_dynamic_max(c)) return cudaErrorInvalidConfiguration;
    if ((e = smem_optin(c, jam_sph_los_kernel)) != cudaSuccess) return e;
    {
        ProfScope ps(c, GK_JAM_SPH_LOS);
        jam_sph_los_kernel<<<dim3((c->nxf * c->nyf + 127) / 128, B), 128, smem2, c->stream>>>(l);
        e = cudaGetLastError();
    }
    return e;
}
