// Row a6 on the 5th-generation tensor cores (tcgen05 + TMEM), the default path of libglad.
//
// Same contraction as jam_quad.cu:  S[iy,ix] = sum_m Y[m,iy] * X[m,ix]  with operands generated on the fly,
// but the operands go from shared memory straight into tcgen05.mma (kind::tf32, fp32 accumulate in TMEM) instead
// of through registers: profiles/r1a.md shows the FP32 SIMT form is bound by shared-memory -> register operand
// delivery (an 8x8 register tile needs one LDS wavefront per FFMA issue slot).
//
// fp32-grade accuracy from TF32 tensor cores: every operand value v is split as v = hi + lo with hi = v rounded
// to TF32 (10-bit mantissa) and lo = v - hi (exact in fp32), and three MMAs are issued per K-step:
//     D += Yhi*Xhi + Yhi*Xlo + Ylo*Xhi            (the dropped lo*lo term is 2^-22 relative)
//
// CTA = (parameter vector, K-slice), 256 threads, all of them operand producers:
//   chunk c (MC contraction rows):  wait until the MMAs that read stage c%2 have completed (mbarrier armed by
//   tcgen05.commit) -> coefficients of chunk c+1 -> operands of chunk c into stage c%2 in the UMMA canonical
//   MN-major no-swizzle layout (8 k-rows x 16 B core matrices) -> fence.proxy.async -> __syncthreads ->
//   one thread issues 3*MC/8 tcgen05.mma and commits.  The tensor core works on chunk c while the CUDA cores
//   produce chunk c+1.  Epilogue: tcgen05.ld the accumulator and write this slice's partial map.
#include "glad_internal.h"

#define LOG2E_F 1.4426950408889634f
#define TC_THREADS 256

struct JTArgs {
    const float* tab; int tabsz; int nl; int nmx;
    const float* un; const float* uw; int nu;
    const float* xf2; const float* yf2; int nxf, nyf;
    int Mpad, Npad;      // UMMA M (64 / 128) and N
    int GX, GY;          // real 4-element groups along x and y: ceil(nxf/4), ceil(nyf/4)
    int MC, lgMC;        // contraction rows per stage (power of two, >= 32)
    int tmem_cols;       // power of two >= 32, >= Npad
    int S;
    float* partial;
};

__device__ __forceinline__ float ex2_tc(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
// UMMA shared-memory descriptor, no swizzle, version 1 (sm_100); SBO = 128 B between 16-byte groups along M/N,
// LBO = byte distance between 8-row K groups (one group per tf32 MMA, so it is never stepped).
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes) {
    uint32_t lo = ((saddr >> 4) & 0x3FFFu) | (((lbo_bytes >> 4) & 0x3FFFu) << 16);
    uint32_t hi = (128u >> 4) | (1u << 14);
    return ((uint64_t)hi << 32) | lo;
}
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// split v = hi + lo, hi on the TF32 grid (round to nearest on the magnitude), lo exact
__device__ __forceinline__ void split_tf32(float v, float& hi, float& lo) {
    hi = __uint_as_float((__float_as_uint(v) + 0x1000u) & 0xFFFFE000u);
    lo = v - hi;
}

__global__ void __launch_bounds__(TC_THREADS) jam_quad_tc_kernel(JTArgs a) {
    extern __shared__ __align__(128) float sm[];
    __shared__ __align__(8) uint64_t s_bar[3];     // empty[0], empty[1], done
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = blockIdx.x / a.S, s = blockIdx.x - b * a.S;
    const float* Tg = a.tab + (size_t)b * a.tabsz;
    if (__float_as_int(Tg[JH_VALID]) == 0) return;

    const int nl = a.nl, nmx = a.nmx, nu = a.nu, MC = a.MC, GX = a.GX, GY = a.GY;
    const int nup = (nu + 1) & ~1;
    // operand stage: [Yhi | Ylo | Xhi | Xlo]; an array holds MC/8 K-steps of G core matrices (8 k-rows x 16 B)
    const int ysz = MC * GY * 4, xsz = MC * (a.Npad >> 2) * 4;   // floats per array
    const int stage_floats = 2 * ysz + 2 * xsz;
    float* s_tab = sm;
    float* s_u2 = s_tab + a.tabsz;
    float* s_wu2 = s_u2 + nup;
    float* s_c2 = s_wu2 + nup;                       // (GY + GX) * 4 squared coordinates, y first
    float* s_coef = s_c2 + (GY + GX) * 4;            // 2 * MC * 4
    float* s_ops = s_coef + 2 * MC * 4;              // 2 stages + tail pad (the M padding rows are read from beyond Y)
    s_ops = (float*)(((uintptr_t)s_ops + 127) & ~(uintptr_t)127);

    for (int i = tid; i < a.tabsz; i += TC_THREADS) s_tab[i] = Tg[i];
    for (int i = tid; i < nu; i += TC_THREADS) { float u = a.un[i]; s_u2[i] = u * u; s_wu2[i] = a.uw[i] * u * u; }
    for (int i = tid; i < (GY + GX) * 4; i += TC_THREADS) {
        float v = 0.f;
        if (i < GY * 4) { if (i < a.nyf) v = a.yf2[i]; }
        else { int j = i - GY * 4; if (j < a.nxf) v = a.xf2[j]; }
        s_c2[i] = v;
    }
    for (int i = tid; i < 2 * stage_floats + 1024; i += TC_THREADS) s_ops[i] = 0.f;   // padding groups stay zero
    if (tid == 0) {
        mbar_init(smem_u32(&s_bar[0]), 1);
        mbar_init(smem_u32(&s_bar[1]), 1);
        mbar_init(smem_u32(&s_bar[2]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        __syncwarp();
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(a.tmem_cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // the zero fill is read by the async proxy
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = s_tmem;

    const float* TL = s_tab + JT_HDR;
    const float* TM = TL + JL_COUNT * nl;
    const float* TC = TM + JM_COUNT * nmx;
    const float* TD = TC + nmx * nl;
    const float cos2i = s_tab[JH_COS2I];
    const int nm = __float_as_int(s_tab[JH_NM]);
    const int pairs = nm * nl;
    const int M = nu * pairs;
    const int NCH = (M + MC - 1) >> a.lgMC;
    const int c0 = (int)(((long)s * NCH) / a.S), c1 = (int)(((long)(s + 1) * NCH) / a.S);

    auto coef = [&](int c, int buf) {
        if (c >= c1) return;
        for (int i = tid; i < MC; i += TC_THREADS) {
            int m = c * MC + i;
            float4 o = make_float4(0.f, 0.f, 0.f, 0.f);      // (P, Q, F0, F1); rows past the end contribute 0
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
    // item e -> (group g = e / MC, row m = e % MC): consecutive lanes take consecutive rows of one group, so the
    // coefficient loads and the 16-byte operand stores of a quarter-warp are contiguous (conflict-free).
    auto produce = [&](int buf) {
        const float4* cf = reinterpret_cast<const float4*>(s_coef) + buf * MC;
        const float4* c2 = reinterpret_cast<const float4*>(s_c2);
        float* st = s_ops + (size_t)buf * stage_floats;
        const int items = MC * (GY + GX);
        for (int e = tid; e < items; e += TC_THREADS) {
            const int g = e >> a.lgMC, m = e & (MC - 1);
            const float4 k = cf[m], q = c2[g];
            float4 v, hi, lo;
            float* dst;
            if (g < GY) {                                    // warp-uniform (MC >= 32)
                const float ne = -k.y;
                v.x = ex2_tc(ne * q.x); v.y = ex2_tc(ne * q.y); v.z = ex2_tc(ne * q.z); v.w = ex2_tc(ne * q.w);
                dst = st + (((m >> 3) * GY + g) * 8 + (m & 7)) * 4;
                split_tf32(v.x, hi.x, lo.x); split_tf32(v.y, hi.y, lo.y); split_tf32(v.z, hi.z, lo.z); split_tf32(v.w, hi.w, lo.w);
                *reinterpret_cast<float4*>(dst) = hi;
                *reinterpret_cast<float4*>(dst + ysz) = lo;
            } else {
                const float ne = -k.x;
                v.x = fmaf(k.w, q.x, k.z) * ex2_tc(ne * q.x);
                v.y = fmaf(k.w, q.y, k.z) * ex2_tc(ne * q.y);
                v.z = fmaf(k.w, q.z, k.z) * ex2_tc(ne * q.z);
                v.w = fmaf(k.w, q.w, k.z) * ex2_tc(ne * q.w);
                dst = st + 2 * ysz + (((m >> 3) * (a.Npad >> 2) + (g - GY)) * 8 + (m & 7)) * 4;
                split_tf32(v.x, hi.x, lo.x); split_tf32(v.y, hi.y, lo.y); split_tf32(v.z, hi.z, lo.z); split_tf32(v.w, hi.w, lo.w);
                *reinterpret_cast<float4*>(dst) = hi;
                *reinterpret_cast<float4*>(dst + xsz) = lo;
            }
        }
    };

    // instruction descriptor: D fp32, A/B tf32, both MN-major, N>>3, M>>4
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 15) | (1u << 16) | ((uint32_t)(a.Npad >> 3) << 17) |
                           ((uint32_t)(a.Mpad >> 4) << 24);
    const uint32_t ops_addr = smem_u32(s_ops);
    const uint32_t ystep = GY * 128, xstep = (a.Npad >> 2) * 128;   // bytes per K-step inside an array

    coef(c0, 0);
    __syncthreads();
    for (int c = c0; c < c1; ++c) {
        const int it = c - c0, buf = it & 1;
        if (it >= 2) mbar_wait(smem_u32(&s_bar[buf]), ((it >> 1) - 1) & 1);   // MMAs of chunk c-2 have read this stage
        coef(c + 1, buf ^ 1);
        produce(buf);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t sb = ops_addr + (uint32_t)buf * stage_floats * 4;
            for (int ks = 0; ks < (MC >> 3); ++ks) {
                const uint64_t yhi = umma_desc(sb + ks * ystep, ystep), ylo = umma_desc(sb + ysz * 4 + ks * ystep, ystep);
                const uint64_t xhi = umma_desc(sb + 2 * ysz * 4 + ks * xstep, xstep);
                const uint64_t xlo = umma_desc(sb + 2 * ysz * 4 + xsz * 4 + ks * xstep, xstep);
                umma_tf32(tmem, yhi, xhi, idesc, (it | ks) ? 1u : 0u);
                umma_tf32(tmem, yhi, xlo, idesc, 1u);
                umma_tf32(tmem, ylo, xhi, idesc, 1u);
            }
            umma_commit(smem_u32(&s_bar[buf]));
            if (c == c1 - 1) umma_commit(smem_u32(&s_bar[2]));
        }
        __syncwarp();
    }

    // epilogue: TMEM -> registers -> this slice's partial map
    const int npf = a.nxf * a.nyf;
    float* out = a.partial + ((size_t)b * a.S + s) * npf;
    if (c1 > c0) {
        mbar_wait(smem_u32(&s_bar[2]), 0);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const int q = warp & 3, half = warp >> 2;                       // lane quarter, column half
        const int row = (a.Mpad == 64) ? (lane < 16 ? 16 * q + lane : -1) : 32 * q + lane;
        for (int cb = half * 8; cb < a.Npad; cb += 16) {
            uint32_t r[8];
            const uint32_t taddr = tmem + ((uint32_t)(32 * q) << 16) + (uint32_t)cb;
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                         : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                         : "r"(taddr));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (row >= 0 && row < a.nyf) {
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (cb + j < a.nxf) out[row * a.nxf + cb + j] = __uint_as_float(r[j]);
            }
        }
    } else {
        for (int i = tid; i < npf; i += TC_THREADS) out[i] = 0.f;
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(a.tmem_cols) : "memory");
}

bool jam_quad_tc_supported(const glad_ctx* c) { return c->nyf <= 128 && c->nxf <= 256; }

cudaError_t launch_jam_quad_tc(glad_ctx* c, int B, int nl, int nmx, int S) {
    JTArgs a;
    a.tab = c->d_jam_tab; a.tabsz = jam_table_floats(nl, nmx); a.nl = nl; a.nmx = nmx;
    a.un = c->d_un; a.uw = c->d_uw; a.nu = c->nu;
    a.xf2 = c->d_xf2; a.yf2 = c->d_yf2; a.nxf = c->nxf; a.nyf = c->nyf;
    a.Mpad = c->nyf <= 64 ? 64 : 128;
    int nalign = a.Mpad == 64 ? 8 : 16;
    a.Npad = ((c->nxf + nalign - 1) / nalign) * nalign;
    a.GX = (c->nxf + 3) / 4; a.GY = (c->nyf + 3) / 4;
    a.tmem_cols = 32;
    while (a.tmem_cols < a.Npad) a.tmem_cols <<= 1;
    a.S = S; a.partial = c->d_partial;
    size_t fixed = (size_t)a.tabsz + 2 * (size_t)((c->nu + 1) & ~1) + (size_t)(a.GX + a.GY) * 4;
    size_t smem = 0;
    for (a.MC = 64, a.lgMC = 6; a.MC >= 32; a.MC >>= 1, --a.lgMC) {
        size_t stage = (size_t)2 * a.MC * a.GY * 4 + (size_t)2 * a.MC * (a.Npad >> 2) * 4;
        smem = sizeof(float) * (fixed + 2 * (size_t)a.MC * 4 + 2 * stage + 1024) + 256;
        if (smem <= 100 * 1024 || a.MC == 32) break;
    }
    if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
    static size_t configured = 0;
    if (smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(jam_quad_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    ProfScope ps(c, GK_JAM_QUAD);
    jam_quad_tc_kernel<<<B * S, TC_THREADS, smem, c->stream>>>(a);
    return cudaGetLastError();
}
