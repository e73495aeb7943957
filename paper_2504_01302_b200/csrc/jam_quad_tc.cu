// Row a6 on the 5th-generation tensor cores (tcgen05 + TMEM), the default path of libglad.
//
// Same contraction as jam_quad.cu:  S[iy,ix] = sum_m Y[m,iy] * X[m,ix]  with operands generated on the fly,
// but the operands go from shared memory straight into tcgen05.mma instead of through registers: profiles/r1a.md
// shows the FP32 SIMT form is bound by shared-memory -> register operand delivery.
//
// fp32-grade accuracy from BF16 tensor-core inputs.  Every operand value v is split into NT bf16 terms
//     v = v1 + v2 (+ v3),   v1 = bf16_rn(v),  v2 = bf16_rn(v - v1),  v3 = bf16_rn(v - v1 - v2)
// (residuals are exact in fp32; NT = 2 keeps 16 mantissa bits, |error| <= 2^-17 |v|, NT = 3 keeps 24).  With
// A = [Y1 ; Y2 ; ..] stacked along M and B = [X1 | X2 | ..] stacked along N, ONE kind::f16 MMA per K = 16 step
// yields every cross product Yi*Xj in its own (row block, column block) of the accumulator; an M <= 128 tile
// costs the same as M = 128, so the split is paid only in N.  The epilogue adds the blocks.  Folded maps whose
// NT row blocks do not fit in M = 128 issue NT MMAs per K-step instead: Yt x [X1 | .. | X(NT-t)], all into the
// same columns (the dropped products are 2^-8NT relative).
//
// The tensor core adds into its fp32 accumulator with TRUNCATION (measured on B200: one accumulator over the
// whole contraction, 3360 K-steps, is biased by -1.4e-4 relative).  So the contraction is cut into groups of
// FL chunks; each group accumulates in its own TMEM buffer (two alternate) and is then added, with ordinary
// round-to-nearest FADDs, into fp32 registers that hold the running map.
//
// Operand layout = UMMA canonical K-major, no swizzle: core matrix = 8 rows (pixels) x 16 bytes (8 consecutive
// contraction rows, an "oct"), 128 contiguous bytes; SBO = 128 B between 8-pixel groups, LBO between the two
// octs of one K = 16 step.  A quarter-warp writes one core matrix with one conflict-free 16-byte store per lane.
//
// CTA = (parameter vector, K-slice), PW producer warps + 1 MMA warp, ONE CTA per SM, no CTA-wide barrier in the
// main loop.  The producer warps form G groups that take the chunks in turn (group g: chunks g, g+G, ..), each
// group into its own operand stage of MC rows.  The groups drift apart, so one group's MUFU-heavy operand loop runs
// beside another group's coefficient rows, accumulator adds and waits (in lock step, two stages of 256 rows shared
// by all warps, the XU pipe limited the operand loops and idled in between: profiles/r2.md).  With MC = the group's
// threads a thread owns one oct over ALL its pixel blocks, so the per-chunk costs (wait, coefficient loads, fence,
// arrive) are paid once per oct and (n_y + n_x)/8 blocks.
//   group g, its i-th chunk c = G i + g (MC contraction rows):  wait until the MMAs that read stage g have completed
//   (mbarrier armed by tcgen05.commit) -> add finished accumulator groups into registers -> the oct's blocks of
//   chunk c into stage g -> fence.proxy.async -> bar.arrive on the stage's "full" named barrier (does not block)
//   -> every R-th chunk one coefficient row of later chunks (in the shadow of the MMAs just released).
//   MMA warp, chunk c (in order):  bar.sync on "full" of stage c%G -> an elected lane issues the MMAs and commits to
//   the stage's "empty" mbarrier.  Its loop body is the latency a group sees between arrive and release, so it is
//   kept short: convergent code, warp-uniform operands, descriptors carried from chunk to chunk.
//
// Tried and measured on C2 (1024 vectors, B200), not kept: the X side factorised as e^{-A x^2} = E1[iu,j](x) G[k](x)
// with G in shared memory cuts the XU pipe from 55 % to 36 % but adds 444 shared-memory load
// wavefronts per 256 rows, and LSU + tensor-core wavefronts then fill 98 % of the shared-memory pipe: 1.94 ms against
// 1.93 without it.  Adding accumulator groups early (before the group's own wait) and two blocks in flight without
// register copies were 2-3 % slower.
#include "glad_internal.h"

#define LOG2E_F 1.4426950408889634f

struct JTArgs {
    const float* tab; int tabsz; int nl; int nmx;
    const float* un; const float* uw; int nu;
    const float* xf2; const float* yf2; int nxf, nyf;
    int ny8, nxp;        // padded map rows (multiple of 8) and columns (multiple of 8 or 16)
    int multi;           // 0: A = [Y1;..;Y_NT] in one M=128 tile;  1: NT MMAs per K-step
    int N;               // accumulator columns = NT * nxp
    int MC, lgMC;        // contraction rows per chunk = per stage (32 .. 256)
    int G, lgG;          // producer groups = operand stages (2, 4 or 8)
    int FL;              // chunks per accumulator group (>= 1)
    int cslots;          // coefficient ring slots: G * (power of two >= NPROD/G/MC + 2), slot = chunk % cslots
    int tmem_cols;       // power of two >= 2 * N
    int S;
    float* partial;
};

__device__ __forceinline__ float ex2_tc(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_approx(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
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
// UMMA shared-memory descriptors are K-major, no swizzle, version 1 (sm_100): SBO = 128 B between 8-row groups along M/N,
// LBO = byte distance between the two 16-byte K halves of a K = 16 (bf16) step; low word = (address >> 4) | (LBO >> 4) << 16,
// high word = (SBO >> 4) | 1 << 14.
// tcgen05.mma from convergent code with warp-uniform operands: one elected lane issues (issued from inside an `if (lane == 0)`
// every MMA costs a 16-instruction broadcast loop).  Descriptors come as their low words plus the common high word: only the
// low word moves from MMA to MMA.
__device__ __forceinline__ void umma_bf16_elect(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t desc_hi, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p, e;\n\t.reg .b64 da, db;\n\telect.sync _|e, 0xffffffff;\n\tsetp.ne.b32 p, %5, 0;\n\t"
                 "mov.b64 da, {%1, %3};\n\tmov.b64 db, {%2, %3};\n\t"
                 "@e tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %4, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(desc_hi), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit_elect(uint32_t bar) {
    asm volatile("{\n\t.reg .pred e;\n\telect.sync _|e, 0xffffffff;\n\t"
                 "@e tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}" ::"r"(bar) : "memory");
}
// {hi: bf16_rn(b), lo: bf16_rn(a)}: element a sits at the lower address
__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    uint32_t d; asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(b), "f"(a)); return d;
}
// packed fp32x2 arithmetic (FMUL2 / FFMA2 / FADD2): one issue slot for two lanes-worth of fp32 work
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpk2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f32x2 ex2_2(f32x2 x) { float a, b; unpk2(x, a, b); return pk2(ex2_tc(a), ex2_tc(b)); }
// a -= bf16 low half of w, b -= bf16 high half of w, exactly (mixed-precision FHFMA.BF16: one issue slot per value,
// no unpacking of the bf16 pair into fp32 registers)
__device__ __forceinline__ void bf16_residual(uint32_t w, float& a, float& b) {
    asm("{\n\t.reg .b16 l, h, m;\n\tmov.b32 {l, h}, %2;\n\tmov.b16 m, 0xBF80;\n\t"
        "fma.rn.f32.bf16 %0, l, m, %0;\n\tfma.rn.f32.bf16 %1, h, m, %1;\n\t}" : "+f"(a), "+f"(b) : "r"(w));
}
// split 4 pairs (the 8 rows of one oct, one pixel) into NT bf16 terms and store one 16-byte core-matrix row per term
template <int NT>
__device__ __forceinline__ void split_store(f32x2 (&v)[4], uint4* dst, int term_stride16) {
    float lo[4], hi[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) unpk2(v[j], lo[j], hi[j]);
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        uint32_t w[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            w[j] = pack_bf16(lo[j], hi[j]);
            if (t + 1 < NT) bf16_residual(w[j], lo[j], hi[j]);
        }
        dst[t * term_stride16] = make_uint4(w[0], w[1], w[2], w[3]);
    }
}
// q = a / d for 0 <= a < 2^24 with inv = 1/d (float): the estimate is off by at most one
__device__ __forceinline__ int div_small(int a, int d, float inv) {
    int q = __float2int_rz(__int2float_rn(a) * inv);
    int r = a - q * d;
    return r < 0 ? q - 1 : (r >= d ? q + 1 : q);
}


__device__ __forceinline__ void bar_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// NT = bf16 terms per operand value, PW = producer warps, NACC = accumulator registers per thread (multiple of 8,
// NACC * PW/4 >= nxp: the NT column blocks [X1 | X2 | ..] of the accumulator are added into the same registers)
template <int NT, int NACC, int PW>
__global__ void __launch_bounds__(PW * 32 + 32, 1) jam_quad_tc_kernel(JTArgs a) {
    constexpr int NPROD = PW * 32, NTHR = NPROD + 32;
    const int G = a.G, GW = PW >> a.lgG, GT = GW * 32;     // producer groups; warps and threads per group
    extern __shared__ __align__(128) float sm[];
    __shared__ __align__(8) uint64_t s_bar[9];     // empty[0 .. G-1], done at [8]
    __shared__ uint32_t s_tmem;
    __shared__ int s_stride[3];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = blockIdx.x / a.S, s = blockIdx.x - b * a.S;
    const float* Tg = a.tab + (size_t)b * a.tabsz;
    if (__float_as_int(Tg[JH_VALID]) == 0) return;      // post kernel never reads this vector's partials

    const int nl = a.nl, nmx = a.nmx, nu = a.nu, MC = a.MC, ny8 = a.ny8, nxp = a.nxp, N = a.N;
    const int nyb = ny8 >> 3, nxb = nxp >> 3;                        // 8-pixel blocks per oct: Y blocks, X blocks
    const int GA = NT * nyb, GB = NT * nxb;                          // core matrices per oct: the NT terms stacked
    const int a16 = (MC >> 3) * GA * 8, b16 = (MC >> 3) * GB * 8;    // 16-byte units per stage
    const int stage16 = a16 + b16;
    // per-vector tables re-laid out for the coefficient rows (one wide load per table and row):
    //   s_lk[k] = (1/s_k^2, b_k-term, S0_k, NKS_k), s_ld[k] = D0_k, s_mj[j] = (1/s_j^2, 1-q_j^2, M_j, 0),
    //   s_jk[j*nl+k] = (C_jk, D_jk), s_uw[iu] = (u^2, w u^2)
    const float* TLg = Tg + JT_HDR;
    const float* TMg = TLg + JL_COUNT * nl;
    const float* TCg = TMg + JM_COUNT * nmx;
    const float* TDg = TCg + nmx * nl;
    float4* s_lk = reinterpret_cast<float4*>(sm);
    float4* s_mj = s_lk + nl;
    float2* s_jk = reinterpret_cast<float2*>(s_mj + nmx);
    float2* s_uw = s_jk + nmx * nl;
    float* s_ld = reinterpret_cast<float*>(s_uw + nu);
    float* s_c2 = s_ld + ((nl + 3) & ~3);            // ny8 + nxp squared coordinates, y first
    // coefficient ring: a.cslots chunks, per chunk [-Q log2e | -P log2e | F0 | F1] x MC floats
    float* s_coef = sm + ((4 * nl + 4 * nmx + 2 * nmx * nl + 2 * nu + ((nl + 3) & ~3) + ny8 + nxp + 31) & ~31);
    uint4* s_ops = reinterpret_cast<uint4*>(s_coef + a.cslots * 4 * MC);   // G stages + tail pad, 128-byte aligned

    for (int k = tid; k < nl; k += NTHR) {
        s_lk[k] = make_float4(TLg[JL_INVS2 * nl + k], TLg[JL_BKQ * nl + k], TLg[JL_S0 * nl + k], TLg[JL_NKS * nl + k]);
        s_ld[k] = TLg[JL_D0 * nl + k];
    }
    for (int j = tid; j < nmx; j += NTHR)
        s_mj[j] = make_float4(TMg[JM_INVS2 * nmx + j], TMg[JM_OMQ2 * nmx + j], TMg[JM_MJ * nmx + j], 0.f);
    for (int i = tid; i < nmx * nl; i += NTHR) s_jk[i] = make_float2(TCg[i], TDg[i]);
    for (int i = tid; i < nu; i += NTHR) { float u = a.un[i]; s_uw[i] = make_float2(u * u, a.uw[i] * u * u); }
    for (int i = tid; i < ny8 + nxp; i += NTHR) {                    // padded pixels: coordinate 0, finite values, never stored
        float v = 0.f;
        if (i < ny8) { if (i < a.nyf) v = a.yf2[i]; }
        else { int j = i - ny8; if (j < a.nxf) v = a.xf2[j]; }
        s_c2[i] = v;
    }
    for (int i = tid; i < G * stage16 + 128; i += NTHR) s_ops[i] = make_uint4(0u, 0u, 0u, 0u);
    if (tid == 0) {
        for (int i = 0; i < 9; ++i) mbar_init(smem_u32(&s_bar[i]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        __syncwarp();
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(a.tmem_cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = s_tmem;

    const int nm = __float_as_int(Tg[JH_NM]);
    const int pairs = nm * nl;
    const int M = nu * pairs;
    const int NCH = (M + MC - 1) >> a.lgMC;
    const int c0 = (int)(((long)s * NCH) / a.S), c1 = (int)(((long)(s + 1) * NCH) / a.S);
    const int nch = c1 - c0;
    const uint32_t dstride = (uint32_t)a.tmem_cols >> 1;                // columns between the two accumulator buffers

    if (warp == PW) {
        // ------------------------------------------------------------------ MMA warp
        // The loop body is the latency between a group's arrive and the release of its stage: everything that can be
        // carried from one chunk to the next is (stage descriptors, accumulator group), no division, no multiply.
        // instruction descriptor: D fp32, A/B bf16, both K-major, M = 128, N>>3 filled per MMA
        const uint32_t idesc_base = (1u << 4) | (1u << 7) | (1u << 10) | (8u << 24);
        const uint32_t ops_addr = smem_u32(s_ops);
        const uint32_t a_lbo = GA * 128, b_lbo = GB * 128;              // bytes between the two octs of a K-step
        // descriptors advance by one K-step (two octs) per MMA and by one stage per chunk: only the 14-bit
        // start-address field (16-byte units) changes
        const uint32_t desc_hi = (128u >> 4) | (1u << 14);              // SBO = 128 B, version 1 (see above)
        const uint32_t ad0 = ((ops_addr >> 4) & 0x3FFFu) | (((a_lbo >> 4) & 0x3FFFu) << 16);
        const uint32_t bd0 = (((ops_addr + a16 * 16) >> 4) & 0x3FFFu) | (((b_lbo >> 4) & 0x3FFFu) << 16);
        const uint32_t ad_step = (2 * a_lbo) >> 4, bd_step = (2 * b_lbo) >> 4;
        const uint32_t idesc1 = idesc_base | ((uint32_t)(N >> 3) << 17);
        const uint32_t bar0 = smem_u32(&s_bar[0]);
        const int nks = MC >> 4;
        uint32_t ad_s = ad0, bd_s = bd0;
        int buf = 0, fl = 0;                                            // stage; chunk within the accumulator group
        uint32_t d = tmem;                                              // warp-uniform
        for (int it = 0; it < nch; ++it) {
            bar_sync(1 + buf, GT + 32);                                 // group it%G has written chunk it into its stage
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            uint32_t accum = fl ? 1u : 0u;
            uint32_t ad = ad_s, bd = bd_s;
            if (!a.multi) {
#pragma unroll 4
                for (int ks = 0; ks < nks; ++ks) {
                    umma_bf16_elect(d, ad, bd, desc_hi, idesc1, accum);
                    accum = 1u; ad += ad_step; bd += bd_step;
                }
            } else {
                for (int ks = 0; ks < nks; ++ks) {
#pragma unroll
                    for (int t = 0; t < NT; ++t) {
                        umma_bf16_elect(d, ad + (uint32_t)((t * nyb * 128) >> 4), bd, desc_hi,
                                        idesc_base | ((uint32_t)(((NT - t) * nxp) >> 3) << 17), accum);
                        accum = 1u;
                    }
                    ad += ad_step; bd += bd_step;
                }
            }
            umma_commit_elect(bar0 + 8 * buf);
            if (it == nch - 1) umma_commit_elect(bar0 + 64);
            ++buf; ad_s += (uint32_t)stage16; bd_s += (uint32_t)stage16;
            if (buf == G) { buf = 0; ad_s = ad0; bd_s = bd0; }
            if (++fl == a.FL) { fl = 0; d = d == tmem ? tmem + dstride : tmem; }
        }
    } else {
        // ------------------------------------------------------------------ producer warps
        const float cos2i = Tg[JH_COS2I];
        const float inv_pairs = 1.f / (float)pairs, inv_nl = 1.f / (float)nl;
        const int grp = warp / GW, lw = warp - grp * GW, lt = tid - grp * GT;   // producer group, warp and thread in it

        // Coefficients of contraction row m = (iu, j, k), k fastest: (-Q log2e, -P log2e, F0, F1); rows past the end have
        // F0 = F1 = 0 and contribute 0.  Chunk `rc` (relative to c0) lives in ring slot rc % cslots, so the groups use
        // alternate slots.  After every R-th chunk of the group (R = GT / MC) ALL its threads write one row each of the
        // group's chunks i+2 .. i+R+1 (i = the chunk just handed to the MMA warp), so the warps of a group stay in step.
        // A chunk is therefore written during iteration <= i'-2 and read during iteration i': the reader has passed
        // the "empty" wait of chunk i'-1, so every thread of the group has arrived on "full" of i'-1, which in program
        // order follows its coefficient writes of iteration i'-2.  While a thread writes in iteration i the slowest
        // warp of the group can still be reading chunk i (the writer passed the "empty" wait of i-1): the group's
        // slots i .. i+R+1 are live, cslots/2 >= R+2.
        // one row from its (iu, j, k): 3 MUFU.RCP + 1 MUFU.RSQ (approx, <= 2 ulp: the operands carry 16 bits)
        auto coef_store = [&](int rc, int r, int iu, int j, int k) {
            float cq = 0.f, cp = 0.f, f0 = 0.f, f1 = 0.f;
            if (iu < nu) {
                const float2 uw = s_uw[iu];
                const float4 mj = s_mj[j];
                const float4 lk = s_lk[k];
                const float2 jk = s_jk[j * nl + k];
                const float d0 = s_ld[k];
                const float u2 = uw.x;
                const float t = mj.y * u2, auj = u2 * mj.x;
                const float gg = 1.f - t;
                const float bb = t * auj * rcp_approx(gg);
                const float A = 0.5f * (auj + lk.x);
                const float Bc = 0.5f * (lk.y + bb);
                const float E = fmaf(Bc, cos2i, A);
                const float D = fmaf(-jk.y, u2, d0);
                const float inv = rsqrt_approx(E * gg) * rcp_approx(fmaf(-jk.x, u2, 1.f));
                const float pref = uw.y * mj.z * inv;
                cp = -A * LOG2E_F;
                cq = -(A * (A + Bc)) * rcp_approx(E) * LOG2E_F;
                f0 = pref * lk.z;
                f1 = pref * lk.w * D;
            }
            float* dst = s_coef + (rc & (a.cslots - 1)) * (4 * MC) + r;
            dst[0] = cq; dst[MC] = cp; dst[2 * MC] = f0; dst[3 * MC] = f1;
        };
        auto coef_row = [&](int rc, int r) {                            // prologue: index split by division
            const int m = (c0 + rc) * MC + r;
            const int iu = div_small(m, pairs, inv_pairs), rem = m - iu * pairs;
            const int j = div_small(rem, nl, inv_nl), k = rem - j * nl;
            coef_store(rc, r, iu, j, k);
        };
        const int R = GT / MC;                                          // thread sets of MC threads in a group
        const int cgrp = lt / MC, crow = lt - cgrp * MC;

        // Quarter-warp = one oct of the chunk (8 contraction rows), lane l8 = pixel within an 8-pixel block.  The
        // thread loads the 8 rows' coefficients once (LDS.128 delivers 512 B per warp whatever the broadcast) and
        // reuses them over its blocks.  With MC = GT a quarter-warp owns its oct's whole block list [Y blocks | X blocks];
        // with smaller chunks the list is cut into NQ = GT / MC contiguous ranges of about equal cost (a Y block is
        // about 20, an X block 21 units); a warp holds one range index ("role") and four octs.  Roles alternate every
        // four warps so that each of the SM's four schedulers (warp % 4) sees every role: the ranges are never equal.
        const int qw = lt >> 3, l8 = lt & 7;
        const int NQ = R;                                               // quarter-warps per oct: 1, 2 or 4
        const bool mix = (GW % (4 * NQ)) == 0;
        const int role = mix ? (lw >> 2) % NQ : lw % NQ;
        const int oct = (qw & 3) + 4 * (mix ? (lw & 3) + 4 * (lw / (4 * NQ)) : lw / NQ);
        int yb0, yb1, xb0, xb1;
        {
            const int ctot = 20 * nyb + 21 * nxb;
            int bnd[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int target = ((role + e) * ctot * 2 + NQ) / (2 * NQ);          // round(role * ctot / NQ)
                int best = 0, bestd = target, pre = 0;
                for (int i = 1; i <= nyb + nxb; ++i) {
                    pre += i <= nyb ? 20 : 21;
                    const int dd = pre > target ? pre - target : target - pre;
                    if (dd < bestd) { bestd = dd; best = i; }
                }
                bnd[e] = (role + e == NQ) ? nyb + nxb : ((role + e == 0) ? 0 : best);
            }
            yb0 = min(bnd[0], nyb); yb1 = min(bnd[1], nyb);
            xb0 = max(bnd[0], nyb) - nyb; xb1 = max(bnd[1], nyb) - nyb;
        }
        // per-thread constants of the block loops: first squared coordinate, first destination row, trip counts
        const float* const qy0 = s_c2 + yb0 * 8 + l8;
        const float* const qx0 = s_c2 + ny8 + xb0 * 8 + l8;
        const int offA = oct * GA * 8 + l8 + yb0 * 8, offB = a16 + oct * GB * 8 + l8 + xb0 * 8;
        const int nyblk = yb1 - yb0, nxblk = xb1 - xb0;
        const int tsA = nyb * 8, tsB = nxb * 8;                          // 16-byte units between the bf16 terms of a value
        auto produce = [&](int rc, int buf) {
            const float* cb = s_coef + (rc & (a.cslots - 1)) * (4 * MC) + 8 * oct;
            uint4* const stage = s_ops + buf * stage16;
            if (nyblk > 0) {
                const float4 e0 = *reinterpret_cast<const float4*>(cb), e1 = *reinterpret_cast<const float4*>(cb + 4);
                const f32x2 c0 = pk2(e0.x, e0.y), c1 = pk2(e0.z, e0.w), c2 = pk2(e1.x, e1.y), c3 = pk2(e1.z, e1.w);
                const float* qp = qy0;
                uint4* dst = stage + offA;
                // software pipeline: the MUFU burst of block n+1 is issued before block n is split and stored, so the
                // XU pipe (4 lanes per scheduler: 8 cycles per warp instruction) works while the warp packs
                auto yvals = [&](const float* p, f32x2 (&v)[4]) {
                    const float q = *p;
                    const f32x2 qq = pk2(q, q);
                    v[0] = ex2_2(mul2(c0, qq)); v[1] = ex2_2(mul2(c1, qq));
                    v[2] = ex2_2(mul2(c2, qq)); v[3] = ex2_2(mul2(c3, qq));
                };
                f32x2 cur[4];
                yvals(qp, cur);
                for (int n = nyblk - 1; n > 0; --n) {
                    f32x2 nxt[4];
                    qp += 8;
                    yvals(qp, nxt);
                    split_store<NT>(cur, dst, tsA);
                    dst += 8;
#pragma unroll
                    for (int j = 0; j < 4; ++j) cur[j] = nxt[j];
                }
                split_store<NT>(cur, dst, tsA);
            }
            if (nxblk > 0) {
                const float* cx = cb + MC;
                const float4 p0 = *reinterpret_cast<const float4*>(cx), p1 = *reinterpret_cast<const float4*>(cx + 4);
                const float4 g0 = *reinterpret_cast<const float4*>(cx + MC), g1 = *reinterpret_cast<const float4*>(cx + MC + 4);
                const float4 h0 = *reinterpret_cast<const float4*>(cx + 2 * MC), h1 = *reinterpret_cast<const float4*>(cx + 2 * MC + 4);
                const float* qp = qx0;
                uint4* dst = stage + offB;
                auto xvals = [&](const float* p, f32x2 (&v)[4]) {
                    const float q = *p;
                    const f32x2 qq = pk2(q, q);
                    v[0] = mul2(fma2(pk2(h0.x, h0.y), qq, pk2(g0.x, g0.y)), ex2_2(mul2(pk2(p0.x, p0.y), qq)));
                    v[1] = mul2(fma2(pk2(h0.z, h0.w), qq, pk2(g0.z, g0.w)), ex2_2(mul2(pk2(p0.z, p0.w), qq)));
                    v[2] = mul2(fma2(pk2(h1.x, h1.y), qq, pk2(g1.x, g1.y)), ex2_2(mul2(pk2(p1.x, p1.y), qq)));
                    v[3] = mul2(fma2(pk2(h1.z, h1.w), qq, pk2(g1.z, g1.w)), ex2_2(mul2(pk2(p1.z, p1.w), qq)));
                };
                f32x2 cur[4];
                xvals(qp, cur);
                for (int n = nxblk - 1; n > 0; --n) {
                    f32x2 nxt[4];
                    qp += 8;
                    xvals(qp, nxt);
                    split_store<NT>(cur, dst, tsB);
                    dst += 8;
#pragma unroll
                    for (int j = 0; j < 4; ++j) cur[j] = nxt[j];
                }
                split_store<NT>(cur, dst, tsB);
            }
        };

        // running map in registers: thread (lane quarter lq, column group cg) holds sum_tc D[32 lq + lane][tc nxp + cg NACC + i]
        float acc[NACC];
#pragma unroll
        for (int i = 0; i < NACC; ++i) acc[i] = 0.f;
        const int lq = warp & 3, cg = warp >> 2;
        auto flush = [&](int g) {
            const uint32_t taddr = tmem + ((uint32_t)(32 * lq) << 16) + (uint32_t)(g & 1) * dstride + (uint32_t)(cg * NACC);
#pragma unroll
            for (int tc = 0; tc < NT; ++tc) {
#pragma unroll
                for (int i = 0; i < NACC; i += 8) {
                    if (cg * NACC + i >= nxp) break;                    // warp-uniform: columns past the term block
                    uint32_t r[8];
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                                 : "r"(taddr + (uint32_t)(tc * nxp + i)));
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int j = 0; j < 8; ++j) acc[i + j] += __uint_as_float(r[j]);
                }
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        };

        // The MMA warp starts chunk c after the MMAs of c-1 .. c-G+1 were issued, i.e. after every other group passed
        // the wait before its latest chunk c' > c-G and added the accumulator groups complete by c'-G >= c-2G+1; this
        // group has added those complete by c-G.  The TMEM buffer that chunk c re-initialises held the accumulator
        // group that ended with chunk c - FL - 1: FL >= 2G - 2.
        int gf = 0;                                                     // next accumulator group to add into acc
        const uint32_t bar_empty = smem_u32(&s_bar[grp]);
        if (tid == 0) {                                                 // the stride NPROD as (du, dj, dk): CTA-uniform, kept in smem
            const int sdu = div_small(NPROD, pairs, inv_pairs), srem = NPROD - sdu * pairs;
            const int sdj = div_small(srem, nl, inv_nl);
            s_stride[0] = sdu; s_stride[1] = sdj; s_stride[2] = srem - sdj * nl;
        }
        if (nch > 0) {
            for (int e = cgrp; e < 2; e += R)                           // the group's first two chunks
                if (grp + G * e < nch) coef_row(grp + G * e, crow);
            bar_sync(9, NPROD);
        }
        int cphase = 0;                                                 // i % R
        // In the loop a thread's rows advance by R chunks of the group = NPROD contraction rows per call: (iu, j, k) is
        // carried, not divided.
        int ciu, cj, ck;
        {
            const int m0 = (c0 + grp + G * (2 + cgrp)) * MC + crow;
            ciu = div_small(m0, pairs, inv_pairs);
            const int rem = m0 - ciu * pairs;
            cj = div_small(rem, nl, inv_nl); ck = rem - cj * nl;
        }
        const int ng = (nch - grp + G - 1) >> a.lgG;                    // chunks of this group
        for (int i = 0; i < ng; ++i) {
            const int rc = grp + G * i;
            if (i >= 1) {
                mbar_wait(bar_empty, (i - 1) & 1);                      // the MMAs of the group's previous chunk are complete
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                while ((gf + 1) * a.FL - 1 <= rc - G) flush(gf++);
            }
            produce(rc, grp);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            bar_arrive(1 + grp, GT + 32);
            if (cphase == 0) {                                          // the group's chunks i+2 .. i+R+1, one row per thread
                const int rcw = rc + G * (2 + cgrp);
                if (rcw < nch) coef_store(rcw, crow, ciu, cj, ck);
                ck += s_stride[2]; if (ck >= nl) { ck -= nl; ++cj; }
                cj += s_stride[1]; if (cj >= nm) { cj -= nm; ++ciu; }
                ciu += s_stride[0];
            }
            cphase = cphase + 1 == R ? 0 : cphase + 1;
        }

        // epilogue: remaining groups -> registers -> shared memory (fold the term blocks) -> this slice's partial map
        const int npf = a.nxf * a.nyf;
        float* out = a.partial + ((size_t)b * a.S + s) * npf;
        if (nch > 0) {
            mbar_wait(smem_u32(&s_bar[8]), 0);                           // all MMAs done: the stages are free
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            while (gf * a.FL < nch) flush(gf++);
            float* scr = reinterpret_cast<float*>(s_ops);                // [128][nxp]
            const int row = 32 * lq + lane;
#pragma unroll
            for (int i = 0; i < NACC; ++i) {
                const int col = cg * NACC + i;
                if (col < nxp) scr[row * nxp + col] = acc[i];
            }
            bar_sync(9, NPROD);
            const int TR = a.multi ? 1 : NT;
            for (int i = tid; i < npf; i += NPROD) {
                const int iy = i / a.nxf, ix = i - iy * a.nxf;
                float v = 0.f;
                for (int tr = TR - 1; tr >= 0; --tr) v += scr[(tr * ny8 + iy) * nxp + ix];   // small terms first
                out[i] = v;
            }
        } else {
            for (int i = tid; i < npf; i += NPROD) out[i] = 0.f;
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(a.tmem_cols) : "memory");
}

// bf16 terms per operand: 2 by default (16 mantissa bits, per-term error <= 2^-16), 3 after glad_set_jam_options(.., 3, ..)
static int tc_terms(const glad_ctx* c) { return c->jam_terms == 3 ? 3 : 2; }
#define TC_PW 16    // producer warps per CTA (24 was tried: 72 registers per thread spill, slower)
#define TC_GROUPS 8 // producer groups = operand stages (measured on C2: 2 -> 2.05 ms, 4 -> 1.97, 8 -> 1.92)

// launch plan for the current sky grid and table sizes; false = not supported (the FP32 kernel takes over)
static bool tc_plan(const glad_ctx* c, int nl, int nmx, JTArgs* a, int* nacc, size_t* smem) {
    const int NT = tc_terms(c), PW = TC_PW;
    a->ny8 = (c->nyf + 7) & ~7;
    if (a->ny8 > 128) return false;
    a->multi = NT * a->ny8 > 128 ? 1 : 0;
    a->nxp = (NT == 3 || a->multi) ? ((c->nxf + 15) & ~15) : ((c->nxf + 7) & ~7);
    a->N = NT * a->nxp;
    if (a->N > 256) return false;
    const int per = (a->nxp + PW / 4 - 1) / (PW / 4);                    // accumulator columns per warp of a lane quarter
    *nacc = per <= 16 ? 16 : (per <= 24 ? 24 : 32);
    a->tmem_cols = 512;                                                  // one CTA per SM: two accumulator buffers of 256 columns
    const size_t fixed = (((size_t)4 * nl + 4 * nmx + 2 * (size_t)nmx * nl + 2 * (size_t)c->nu + ((nl + 3) & ~3) +
                           (size_t)(a->ny8 + a->nxp) + 31) & ~(size_t)31) * 4;
    // RT = contraction rows in flight (all stages): with RT = producer threads a quarter-warp owns its oct's whole
    // block list; each halving doubles the quarter-warps per oct
    for (int RT = PW * 32; RT >= PW * 8; RT >>= 1) {
        a->G = TC_GROUPS;
        while (RT / a->G < 32) a->G >>= 1;                                   // a warp's quarters take 4 different octs of a chunk
        for (a->lgG = 0; (1 << a->lgG) < a->G; ++a->lgG) {}
        a->MC = RT >> a->lgG;
        for (a->lgMC = 0; (1 << a->lgMC) < a->MC; ++a->lgMC) {}
        size_t ops = (size_t)RT * NT * (a->ny8 + a->nxp) * 2 + 2048;         // G stages + the M = 128 over-read
        const size_t scr = (size_t)128 * a->nxp * 4;                         // epilogue scratch reuses the stages
        if (ops < scr) ops = scr;
        const int R = PW * 32 / RT;                                          // group threads / MC
        a->cslots = a->G * (R <= 2 ? 4 : 8);                                 // G * pow2(R + 2)
        *smem = fixed + (size_t)a->cslots * 4 * a->MC * 4 + ops;
        if (*smem <= 225 * 1024) return true;
    }
    return false;
}

bool jam_quad_tc_supported(const glad_ctx* c, int nl, int nmx) { JTArgs a; int nacc; size_t smem; return tc_plan(c, nl, nmx, &a, &nacc, &smem); }

template <int NT, int NACC, int PW>
static cudaError_t tc_launch(const glad_ctx* c, const JTArgs& a, int grid, size_t smem, cudaStream_t st) {
    cudaError_t e = smem_optin(c, jam_quad_tc_kernel<NT, NACC, PW>);
    if (e != cudaSuccess) return e;
    jam_quad_tc_kernel<NT, NACC, PW><<<grid, PW * 32 + 32, smem, st>>>(a);
    return cudaGetLastError();
}
template <int NT>
static cudaError_t tc_dispatch(const glad_ctx* c, const JTArgs& a, int nacc, int grid, size_t smem, cudaStream_t st) {
    if (nacc == 16) return tc_launch<NT, 16, 16>(c, a, grid, smem, st);
    if (nacc == 24) return tc_launch<NT, 24, 16>(c, a, grid, smem, st);
    return tc_launch<NT, 32, 16>(c, a, grid, smem, st);
}

cudaError_t launch_jam_quad_tc(glad_ctx* c, int B, int nl, int nmx, int S) {
    JTArgs a;
    int nacc;
    size_t smem;
    if (!tc_plan(c, nl, nmx, &a, &nacc, &smem)) return cudaErrorInvalidConfiguration;
    a.tab = c->d_jam_tab; a.tabsz = jam_table_floats(nl, nmx); a.nl = nl; a.nmx = nmx;
    a.un = c->d_un; a.uw = c->d_uw; a.nu = c->nu;
    a.xf2 = c->d_xf2; a.yf2 = c->d_yf2; a.nxf = c->nxf; a.nyf = c->nyf;
    a.S = S; a.partial = c->d_partial;
    // 512 contraction rows (32 K-steps) per accumulator group, but not fewer chunks than the kernel's TMEM buffer
    // reuse argument needs (2G - 2)
    a.FL = 512 / a.MC;
    if (c->jam_flush >= 1) a.FL = c->jam_flush;
    if (a.FL < 2 * a.G - 2) a.FL = 2 * a.G - 2;
    ProfScope ps(c, GK_JAM_QUAD);
    return tc_terms(c) == 3 ? tc_dispatch<3>(c, a, nacc, B * S, smem, c->stream) : tc_dispatch<2>(c, a, nacc, B * S, smem, c->stream);
}
