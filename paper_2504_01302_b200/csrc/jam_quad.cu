// Row a6 of SURVEY.md 8(a): the JAM quadrature, the dominant cost of the joint likelihood.
//
// For one parameter vector the map is  S[iy,ix] = sum_m Y[m,iy] * X[m,ix],  m = (node u, mass Gaussian j,
// luminous Gaussian k), because in the R-D1 formula the sky pixel enters each term only through
//     (F0_m + F1_m x'^2) exp(-P_m x'^2) * exp(-Q_m y'^2)
// and the sky grid is a tensor product x'[ix] x y'[iy] (R-D5).  This is a dense contraction over
// K = nu*nm*nl (5e4 .. 2.4e5) whose operands are GENERATED ON THE FLY and never exist in HBM:
//     X[m,ix] = (F0_m + F1_m x2) 2^(-P_m x2),   Y[m,iy] = 2^(-Q_m y2)          (P, Q pre-multiplied by log2 e)
// so the exponentials drop from nx*ny to nx+ny per term and the rest is FP32 FFMA on an 8x8 register tile.
// When the grid is mirror-symmetric only the folded half per axis is computed (the integrand is even).
//
// One CTA = (parameter vector b, K-slice s).  Threads form NG groups of G = tiles-per-map threads; every group
// owns the whole (folded) map as 8x8 register tiles and consumes its own rows of each staged chunk of
// MC = NG*JQ_MI contraction rows.  Software pipeline per chunk c (one __syncthreads each):
//     coefficients of chunk c+2  ->  operands of chunk c+1 (MUFU.EX2)  ->  FFMA over chunk c.
#include "glad_internal.h"

#define LOG2E_F 1.4426950408889634f

struct JQArgs {
    const float* tab; int tabsz; int nl; int nmx;
    const float* un; const float* uw; int nu;
    const float* xf2; const float* yf2; int nxf, nyf;
    int tnx, tny, G, NG, S;
    float* partial;
};

__device__ __forceinline__ float ex2_fast(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__global__ void __launch_bounds__(512, 1) jam_quad_kernel(JQArgs a) {
    extern __shared__ __align__(16) float sm[];
    const int tid = threadIdx.x, NT = blockDim.x;
    const int b = blockIdx.x / a.S, s = blockIdx.x - b * a.S;
    const float* Tg = a.tab + (size_t)b * a.tabsz;
    if (__float_as_int(Tg[JH_VALID]) == 0) return;      // post kernel never reads this vector's partials

    const int nl = a.nl, nmx = a.nmx, nu = a.nu;
    const int nxp = a.tnx * JQ_T, nyp = a.tny * JQ_T, RS = nxp + nyp, RS4 = RS >> 2;
    const int MC = a.NG * JQ_MI;
    const int opsz = max(2 * MC * RS, nxp * nyp);
    float* s_tab = sm;                       // tabsz
    const int nup = (nu + 1) & ~1;           // keeps the float4 regions 16-byte aligned
    float* s_u2 = s_tab + a.tabsz;           // nup
    float* s_wu2 = s_u2 + nup;               // nup
    float* s_c2 = s_wu2 + nup;               // RS  squared coordinates in operand-row layout
    float* s_coef = s_c2 + RS;               // 2 * MC * 4
    float* s_ops = s_coef + 2 * MC * 4;      // opsz
    (void)opsz;

    for (int i = tid; i < a.tabsz; i += NT) s_tab[i] = Tg[i];
    for (int i = tid; i < nu; i += NT) { float u = a.un[i]; s_u2[i] = u * u; s_wu2[i] = a.uw[i] * u * u; }
    // operand row layout: [X lo (tnx x 4) | X hi (tnx x 4) | Y lo (tny x 4) | Y hi (tny x 4)], tile t holds columns
    // t*8 .. t*8+7 split into a lo and a hi float4 so that a quarter-warp's LDS.128 hits distinct banks.
    for (int c = tid; c < RS; c += NT) {
        float v;
        if (c < nxp) {
            int half = c / (nxp >> 1), r = c - half * (nxp >> 1);
            int ix = (r >> 2) * JQ_T + half * 4 + (r & 3);
            v = ix < a.nxf ? a.xf2[ix] : 0.f;          // padded columns: harmless finite garbage, never stored
        } else {
            int cc = c - nxp;
            int half = cc / (nyp >> 1), r = cc - half * (nyp >> 1);
            int iy = (r >> 2) * JQ_T + half * 4 + (r & 3);
            v = iy < a.nyf ? a.yf2[iy] : 0.f;
        }
        s_c2[c] = v;
    }
    __syncthreads();

    const float* TL = s_tab + JT_HDR;
    const float* TM = TL + JL_COUNT * nl;
    const float* TC = TM + JM_COUNT * nmx;
    const float* TD = TC + nmx * nl;
    const float cos2i = s_tab[JH_COS2I];
    const int nm = __float_as_int(s_tab[JH_NM]);
    const int pairs = nm * nl;
    const int M = nu * pairs;
    const int NCH = (M + MC - 1) / MC;
    const int c0 = (int)(((long)s * NCH) / a.S), c1 = (int)(((long)(s + 1) * NCH) / a.S);

    // consumer role
    const bool active = tid < a.NG * a.G;
    const int g = tid / a.G, r = tid - g * a.G;
    const int ty = r / a.tnx, tx = r - ty * a.tnx;
    const int offXlo = tx * 4, offXhi = (nxp >> 1) + tx * 4, offYlo = nxp + ty * 4, offYhi = nxp + (nyp >> 1) + ty * 4;
    float acc[JQ_T][JQ_T];
#pragma unroll
    for (int i = 0; i < JQ_T; ++i)
#pragma unroll
        for (int j = 0; j < JQ_T; ++j) acc[i][j] = 0.f;

    auto coef = [&](int c, int buf) {
        if (c >= c1) return;
        for (int i = tid; i < MC; i += NT) {
            int m = c * MC + i;
            float4 o = make_float4(0.f, 0.f, 0.f, 0.f);      // (P, Q, F0, F1)
            if (m < M) {
                int iu = m / pairs, rem = m - iu * pairs;
                int j = rem / nl, k = rem - j * nl;
                float u2 = s_u2[iu];
                float omq2 = TM[JM_OMQ2 * nmx + j];
                float auj = u2 * TM[JM_INVS2 * nmx + j];
                float gg = 1.f - omq2 * u2;
                float bb = omq2 * u2 * auj / gg;
                float A = 0.5f * (auj + TL[JL_INVS2 * nl + k]);
                float Bc = 0.5f * (TL[JL_BKQ * nl + k] + bb);
                float E = fmaf(Bc, cos2i, A);
                float D = fmaf(-TD[j * nl + k], u2, TL[JL_D0 * nl + k]);
                float inv = rsqrtf(E * gg) / (1.f - TC[j * nl + k] * u2);
                float pref = s_wu2[iu] * TM[JM_MJ * nmx + j] * inv;
                o.x = A * LOG2E_F;
                o.y = A * (A + Bc) / E * LOG2E_F;
                o.z = pref * TL[JL_S0 * nl + k];
                o.w = pref * TL[JL_NKS * nl + k] * D;
            }
            reinterpret_cast<float4*>(s_coef)[buf * MC + i] = o;
        }
    };
    const float invRS4 = 1.f / (float)RS4;
    const int nx4 = nxp >> 2;
    auto produce = [&](int c, int buf) {
        if (c >= c1) return;
        const float4* cf = reinterpret_cast<const float4*>(s_coef) + buf * MC;
        float4* dst = reinterpret_cast<float4*>(s_ops) + (size_t)buf * MC * RS4;
        const float4* c2 = reinterpret_cast<const float4*>(s_c2);
        for (int e = tid; e < MC * RS4; e += NT) {
            int m = __float2int_rz(((float)e + 0.5f) * invRS4);
            int c4 = e - m * RS4;
            float4 k = cf[m], q = c2[c4], o;
            bool isx = c4 < nx4;
            float ne = isx ? -k.x : -k.y;
            float f0 = isx ? k.z : 1.f, f1 = isx ? k.w : 0.f;
            o.x = fmaf(f1, q.x, f0) * ex2_fast(ne * q.x);
            o.y = fmaf(f1, q.y, f0) * ex2_fast(ne * q.y);
            o.z = fmaf(f1, q.z, f0) * ex2_fast(ne * q.z);
            o.w = fmaf(f1, q.w, f0) * ex2_fast(ne * q.w);
            dst[e] = o;
        }
    };

    coef(c0, 0);
    __syncthreads();
    coef(c0 + 1, 1);
    produce(c0, 0);
    __syncthreads();
    for (int c = c0; c < c1; ++c) {
        const int cur = (c - c0) & 1;
        coef(c + 2, cur);
        produce(c + 1, cur ^ 1);
        if (active) {
            const float* rows = s_ops + (size_t)cur * MC * RS + (size_t)(g * JQ_MI) * RS;
#pragma unroll
            for (int i = 0; i < JQ_MI; ++i) {
                const float* row = rows + i * RS;
                float4 xl = *reinterpret_cast<const float4*>(row + offXlo);
                float4 xh = *reinterpret_cast<const float4*>(row + offXhi);
                float4 yl = *reinterpret_cast<const float4*>(row + offYlo);
                float4 yh = *reinterpret_cast<const float4*>(row + offYhi);
                const float xv[8] = {xl.x, xl.y, xl.z, xl.w, xh.x, xh.y, xh.z, xh.w};
                const float yv[8] = {yl.x, yl.y, yl.z, yl.w, yh.x, yh.y, yh.z, yh.w};
#pragma unroll
                for (int p = 0; p < JQ_T; ++p)
#pragma unroll
                    for (int q = 0; q < JQ_T; ++q) acc[p][q] = fmaf(yv[p], xv[q], acc[p][q]);
            }
        }
        __syncthreads();
    }

    // reduce the NG groups into one tile (fixed order -> deterministic), then write this slice's partial map
    float* tile = s_ops;
    for (int g0 = 0; g0 < a.NG; ++g0) {
        if (active && g == g0) {
#pragma unroll
            for (int p = 0; p < JQ_T; ++p) {
                float* t = tile + (ty * JQ_T + p) * nxp + tx * JQ_T;
#pragma unroll
                for (int q = 0; q < JQ_T; ++q) t[q] = (g0 == 0) ? acc[p][q] : t[q] + acc[p][q];
            }
        }
        __syncthreads();
    }
    const int npf = a.nxf * a.nyf;
    float* out = a.partial + ((size_t)b * a.S + s) * npf;
    for (int i = tid; i < npf; i += NT) {
        int fy = i / a.nxf, fx = i - fy * a.nxf;
        out[i] = tile[fy * nxp + fx];
    }
}

int jam_quad_geometry(const glad_ctx* c, int* groups) {
    int tnx = (c->nxf + JQ_T - 1) / JQ_T, tny = (c->nyf + JQ_T - 1) / JQ_T;
    int G = tnx * tny;
    if (G > 512) return -1;
    int NG = 256 / G;
    if (NG < 1) NG = 1;
    if (NG > 16) NG = 16;
    *groups = NG;
    return ((NG * G + 31) / 32) * 32;
}

cudaError_t launch_jam_quad(glad_ctx* c, int B, int nl, int nmx, int S) {
    JQArgs a;
    a.tab = c->d_jam_tab; a.tabsz = jam_table_floats(nl, nmx); a.nl = nl; a.nmx = nmx;
    a.un = c->d_un; a.uw = c->d_uw; a.nu = c->nu;
    a.xf2 = c->d_xf2; a.yf2 = c->d_yf2; a.nxf = c->nxf; a.nyf = c->nyf;
    a.tnx = (c->nxf + JQ_T - 1) / JQ_T; a.tny = (c->nyf + JQ_T - 1) / JQ_T; a.G = a.tnx * a.tny;
    int NT = jam_quad_geometry(c, &a.NG);
    if (NT < 0) return cudaErrorInvalidConfiguration;
    a.S = S; a.partial = c->d_partial;
    int nxp = a.tnx * JQ_T, nyp = a.tny * JQ_T, RS = nxp + nyp, MC = a.NG * JQ_MI;
    size_t ops = (size_t)2 * MC * RS;
    if ((size_t)nxp * nyp > ops) ops = (size_t)nxp * nyp;
    size_t smem = sizeof(float) * ((size_t)a.tabsz + 2 * (size_t)((c->nu + 1) & ~1) + RS + 2 * (size_t)MC * 4 + ops);
    if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = smem_optin(c, jam_quad_kernel);
    if (e != cudaSuccess) return e;
    ProfScope ps(c, GK_JAM_QUAD);
    jam_quad_kernel<<<B * S, NT, smem, c->stream>>>(a);
    return cudaGetLastError();
}
