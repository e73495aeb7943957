// The contraction of the pixelated-source likelihood on the 5th-generation tensor cores:
//     F = f^T C_d^-1 f  (Eq. 41),  D = f^T C_d^-1 d  (Eq. 42),   f = B L  [N_pix, N_s] fp32 in HBM
// A genuine dense contraction over the image pixels (K = N_pix ~ 1e4, M = N = N_s ~ 1e3; Table 1), so it runs as
// tcgen05.mma with the accumulator in TMEM.  fp32-grade results from 16-bit inputs by splitting, as in jam_quad_tc.cu, but into
// FP16 terms: F + lambda g has condition numbers of 1e5-1e6, and with two bf16 terms (16 mantissa bits) the source pixels and the
// model at masked image pixels came out 2.5e-4 off (measured; the fp32 SIMT kernel this replaces gave 1e-6).  Two fp16 terms keep
// 22 bits: v1 = fp16_rn(v), v2 = fp16_rn(v - v1).  fp16 has 5 exponent bits, so both operands are first scaled by exact powers of
// two (from max ivar and sum |psf|, static data) to sit just below 2^14, and the tile is scaled back in the epilogue.  Three
// products are issued,
//     D[128 x 256] += A1 x [B1 | B2]   (hi.hi in columns 0..127, hi.lo in 128..255),   D[:, 0..127] += A2 x B1   (lo.hi),
// A = (ivar f)^T tile (the weight goes into one side only), B = f tile; the lo.lo product (2^-22 relative) is dropped.  The
// tensor core adds into TMEM with truncation, so the K loop is cut into groups of SY_FL chunks (512 pixels) that alternate between
// two TMEM buffers and are added into fp32 registers with ordinary round-to-nearest FADDs.
//
// CTA = (vector, 128 x 128 output tile of the lower triangle), 512 threads, one CTA per SM.  A pre-pass lists the image pixels that
// count for the tile (the f row touches both column blocks: the PSF footprint recorded by the blur kernel) -- about a third of them;
// the sum over pixels can be taken in any order, so only the listed rows are contracted, 32 at a time ("chunk"; skipping whole
// chunks of consecutive pixels instead removes only ~45 %).  The raw fp32 columns of a chunk are gathered into a 3-slot ring by cp.async
// two chunks ahead (the first version loaded them into registers at the point of use: 33 ms per 296 vectors, latency-bound with
// 16 warps per SM).  All threads then convert: thread = (side A/B, column, half of the chunk's pixel octs) reads its 8 pixels of one
// column from the ring (conflict-free), applies ivar (A side), splits, and writes one 16-byte core-matrix row per term into the
// UMMA K-major no-swizzle layout (core matrix = 8 columns x 8 pixels; a warp writes 512 contiguous bytes).  One thread issues the
// MMAs of a chunk and commits them to the stage's mbarrier; the tensor core works on chunk n while the CUDA cores convert n + 1.
// On diagonal tiles the A-side threads also accumulate D (fp64), so f is not read a second time for the right-hand side.
#include "glad_internal.h"
#include "pixsrc_common.cuh"

#define SY_T 128                 // output tile (rows = columns of f on the A side, columns = columns of f on the B side)
#define SY_KC 32                 // image pixels per chunk = 2 MMA K-steps of 16
#define SY_FL 16                 // chunks per TMEM accumulator group (512 pixels)
#define SY_RAW 3                 // ring of raw fp32 chunks (cp.async runs two chunks ahead)
#define SY_RAW_BYTES (2 * SY_KC * SY_T * 4)      // A-side and B-side columns of one chunk: 32 KB
#define SY_THREADS 512
#define SY_A_BYTES (SY_T * SY_KC * 2)            // one bf16 term of the A tile: 16 KB
#define SY_B_BYTES (2 * SY_T * SY_KC * 2)        // [B1 | B2]: 32 KB
#define SY_STAGE_BYTES (2 * SY_A_BYTES + SY_B_BYTES)

__device__ __forceinline__ void px_cp_async16(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ uint32_t sy_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sy_mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void sy_mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
// UMMA shared-memory descriptor: K-major, no swizzle (sm_100 version 1): SBO = 128 B between 8-row groups along M/N, LBO = distance
// between the two 8-element K halves of a K = 16 step
__device__ __forceinline__ uint64_t sy_desc(uint32_t saddr, uint32_t lbo_bytes) {
    const uint32_t lo = ((saddr >> 4) & 0x3FFFu) | (((lbo_bytes >> 4) & 0x3FFFu) << 16);
    const uint32_t hi = (128u >> 4) | (1u << 14);
    return ((uint64_t)hi << 32) | lo;
}
__device__ __forceinline__ void sy_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// One lane of converged warp 0 issues: behind an elect.sync branch ptxas moves the operands into uniform registers with plain R2URs
// (under `if (tid == 0)` every tcgen05.mma is wrapped in a 16-instruction broadcast loop), and descriptors go in as low words plus
// the common high word.  With the CTA-wide barrier still in place this was slower (16.7 against 16.1 ms); now that warp 0 alone
// waits and issues, its own time per chunk is what counts: 14.4 -> 14.0 ms.
__device__ __forceinline__ bool sy_elect_one() {
    uint32_t e;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(e));
    return e != 0;
}
__device__ __forceinline__ void sy_mma_lo(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t desc_hi, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\tsetp.ne.b32 p, %5, 0;\n\t"
                 "mov.b64 da, {%1, %3};\n\tmov.b64 db, {%2, %3};\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %4, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(desc_hi), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void sy_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ uint32_t sy_pack(float a, float b) {        // {hi: fp16(b), lo: fp16(a)}: a at the lower address
    uint32_t d; asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(b), "f"(a)); return d;
}
__device__ __forceinline__ void sy_residual(uint32_t w, float& a, float& b) {   // a -= fp16 lo half of w, b -= hi half, exactly (FHFMA)
    asm("{\n\t.reg .b16 l, h, m;\n\tmov.b32 {l, h}, %2;\n\tmov.b16 m, 0xBC00;\n\t"
        "fma.rn.f32.f16 %0, l, m, %0;\n\tfma.rn.f32.f16 %1, h, m, %1;\n\t}" : "+f"(a), "+f"(b) : "r"(w));
}
// split the 8 pixels of one column into two fp16 terms: one 16-byte core-matrix row each
__device__ __forceinline__ void sy_split(float (&v)[8], uint4& hi, uint4& lo) {
    uint32_t h[4], l[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        h[j] = sy_pack(v[2 * j], v[2 * j + 1]);
        sy_residual(h[j], v[2 * j], v[2 * j + 1]);
        l[j] = sy_pack(v[2 * j], v[2 * j + 1]);
    }
    hi = make_uint4(h[0], h[1], h[2], h[3]);
    lo = make_uint4(l[0], l[1], l[2], l[3]);
}

__global__ void __launch_bounds__(SY_THREADS, 1) pixsrc_syrk_tc_kernel(const float* __restrict__ f, const float* __restrict__ ivar,
                                                                      const float* __restrict__ data, const int2* __restrict__ rng,
                                                                      const float* __restrict__ lam_reg, const double* __restrict__ stat,
                                                                      int npix, int ns, int nsx, int nsy, unsigned short* __restrict__ rowlist,
                                                                      double* __restrict__ A, double* __restrict__ Dv) {
    extern __shared__ __align__(128) unsigned char sy_sm[];
    __shared__ __align__(8) uint64_t s_bar[3];           // stage 0, stage 1, done
    __shared__ uint32_t s_tmem;
    __shared__ float s_w[SY_THREADS / 32][SY_RAW][16], s_wd[SY_THREADS / 32][SY_RAW][16];   // per warp: sA * ivar, ivar * data of its 16 rows
    __shared__ int s_cnt[SY_THREADS / 32], s_nrows;
    __shared__ double s_d[2 * SY_T];
    const int b = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    int ti = (int)((sqrtf(8.f * (float)blockIdx.x + 1.f) - 1.f) * 0.5f);
    while ((ti + 1) * (ti + 2) / 2 <= (int)blockIdx.x) ++ti;
    while (ti * (ti + 1) / 2 > (int)blockIdx.x) --ti;
    const int tj = blockIdx.x - ti * (ti + 1) / 2;
    const int i0 = ti * SY_T, j0 = tj * SY_T;
    const bool diag = ti == tj;
    const float* fb = f + (size_t)b * npix * ns;
    const int2* rb = rng + (size_t)b * npix;

    if (tid == 0) {
        sy_mbar_init(sy_smem_u32(&s_bar[0]), 1);
        sy_mbar_init(sy_smem_u32(&s_bar[1]), 1);
        sy_mbar_init(sy_smem_u32(&s_bar[2]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        __syncwarp();
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sy_smem_u32(&s_tmem)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = s_tmem;

    // producer role: side 0 = A (weighted), 1 = B; column c of the tile; octs og*2, og*2+1 of every chunk
    const int side = (tid >> 7) & 1, c = tid & 127, og = tid >> 8;
    // byte offset of this thread's 16-byte row inside a K-half of its operand (8-row groups are 128 B apart)
    const uint32_t row_off = (uint32_t)((c >> 3) * 128 + (c & 7) * 16);
    double dsum = 0.0;                                   // D of column i0 + c (A side of diagonal tiles)
    // exact power-of-two scales: |f| <= sum |psf| and ivar |f| <= max ivar sum |psf| land in [2^13, 2^14)
    int eb, ea;
    frexp(stat[3], &eb);
    frexp(stat[2] * stat[3], &ea);
    const float sB = ldexpf(1.f, 14 - eb), sA = ldexpf(1.f, 14 - ea), unscale = ldexpf(1.f, ea + eb - 28);

    // running 128 x 128 tile in registers: thread (lane quarter warp % 4, column quarter warp / 4) holds row 32 (warp % 4) + lane,
    // columns 32 (warp / 4) .. + 31, hi.hi + lo.hi + hi.lo added
    float acc[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) acc[i] = 0.f;
    const int lq = warp & 3, cq = warp >> 2;
    auto flush = [&](int g) {
        const uint32_t taddr = tmem + ((uint32_t)(32 * lq) << 16) + (uint32_t)(g & 1) * 256u + (uint32_t)(cq * 32);
#pragma unroll
        for (int half = 0; half < 2; ++half)
#pragma unroll
            for (int i = 0; i < 32; i += 16) {
                uint32_t r[16];
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                             : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                               "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                             : "r"(taddr + (uint32_t)(half * 128 + i)));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int j = 0; j < 16; ++j) acc[i + j] += __uint_as_float(r[j]);
            }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    };

    // instruction descriptor: D fp32 (bit 4), A/B fp16 (format fields 0), both K-major, M = 128; N = 256 or 128
    const uint32_t idesc_base = (1u << 4) | (8u << 24);
    const uint32_t idesc256 = idesc_base | ((256u >> 3) << 17), idesc128 = idesc_base | ((128u >> 3) << 17);
    const uint32_t sm_base = sy_smem_u32(sy_sm);

    // ---- which image pixels count for this tile?  (ivar != 0 and the f row touches both column blocks: about a third of them.)  The
    // contraction is a sum over pixels in any order, so the rows that count are COMPACTED: listed in ascending order (two passes per
    // warp over its segment of the image: count, then write at the prefix offset) and consumed SY_KC at a time.
    unsigned short* list = rowlist + ((size_t)b * gridDim.x + blockIdx.x) * npix;
    {
        const int seg = (((npix + SY_THREADS / 32 - 1) / (SY_THREADS / 32)) + 31) & ~31;
        const int pa = warp * seg, pb = min(npix, pa + seg);
        auto hits = [&](int p) -> bool {
            if (p >= pb) return false;
            const int2 r = rb[p];
            return ivar[p] != 0.f && r.x <= i0 + SY_T - 1 && r.y >= i0 && r.x <= j0 + SY_T - 1 && r.y >= j0;
        };
        int cnt = 0;
        for (int p = pa; p < pb; p += 32) cnt += __popc(__ballot_sync(0xffffffffu, hits(p + lane)));
        if (lane == 0) s_cnt[warp] = cnt;
        __syncthreads();
        int off = 0;
        for (int w = 0; w < warp; ++w) off += s_cnt[w];
        for (int p = pa; p < pb; p += 32) {
            const bool h = hits(p + lane);
            const unsigned m = __ballot_sync(0xffffffffu, h);
            if (h) list[off + __popc(m & ((1u << lane) - 1u))] = (unsigned short)(p + lane);
            off += __popc(m);
        }
        if (tid == SY_THREADS - 1) s_nrows = off;
        __syncthreads();                                 // also makes the list (global memory, written by this CTA) visible to the CTA
    }
    const int nrows = s_nrows, nrel = (nrows + SY_KC - 1) / SY_KC;

    // ---- raw fp32 tiles of f: ring of SY_RAW chunks filled by cp.async two chunks ahead of the conversion.  Every WARP copies
    // exactly the 16 pixel rows x 32 columns it converts (four 16-byte pieces per lane), so a __syncwarp orders copy and use and the
    // ring needs no CTA-wide barrier.
    unsigned char* raw_base = sy_sm + 2 * (size_t)SY_STAGE_BYTES;
    const bool vec4 = (ns & 3) == 0;
    const int col0 = (side ? j0 : i0) + 32 * (warp & 3);                 // first column of this warp
    // the lane's four pieces: fixed (row of the chunk, 4-column segment) inside the warp's block.  A chunk row past the end of the
    // list is read from pixel 0 with A-side weight 0, so it adds nothing.
    int prow[4], pcol[4];
    unsigned fastmask = 0;
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const int piece = lane + 32 * it;
        prow[it] = piece >> 3;                           // 0..15 within the warp's 16 rows
        pcol[it] = col0 + (piece & 7) * 4;
        if (vec4 && pcol[it] + 3 < ns) fastmask |= 1u << it;
    }
    float* const raw_warp = reinterpret_cast<float*>(raw_base) + (side * SY_KC + og * 16) * SY_T + 32 * (warp & 3);
    auto stage_raw = [&](int idx) {                      // rows idx*SY_KC.. of the list -> ring slot idx % SY_RAW (idx >= nrel: nothing)
        if (idx < nrel) {
            const int slot = idx % SY_RAW;
            const int li = idx * SY_KC + og * 16 + (lane & 15);              // lanes 0..15 (and 16..31 again): the warp's 16 rows
            const bool have = li < nrows;
            const int pid = have ? (int)list[li] : 0;
            float* rawp = raw_warp + (size_t)slot * (SY_RAW_BYTES / 4);
#pragma unroll
            for (int it = 0; it < 4; ++it) {
                const int pp = __shfl_sync(0xffffffffu, pid, prow[it]);
                float* dst = rawp + prow[it] * SY_T + (pcol[it] - col0);
                const float* src = fb + (size_t)pp * ns + pcol[it];
                if (fastmask & (1u << it)) px_cp_async16(dst, src);
                else {
                    float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (pcol[it] < ns) z.x = src[0];
                    if (pcol[it] + 1 < ns) z.y = src[1];
                    if (pcol[it] + 2 < ns) z.z = src[2];
                    if (pcol[it] + 3 < ns) z.w = src[3];
                    *reinterpret_cast<float4*>(dst) = z;
                }
            }
            if (side == 0 && lane < 16) {
                const float w = have ? ivar[pid] : 0.f;
                s_w[warp][slot][lane] = w * sA;
                s_wd[warp][slot][lane] = (diag && have) ? w * data[pid] : 0.f;
            }
        }
        asm volatile("cp.async.commit_group;\n" ::: "memory");
    };
    stage_raw(0);
    stage_raw(1);

    int gf = 0;                                          // next accumulator group to add into the registers
    for (int n = 0; n < nrel; ++n) {
        stage_raw(n + 2);                                // slot (n + 2) % 3 was last read while chunk n - 1 was converted
        asm volatile("cp.async.wait_group 2;\n" ::: "memory");
        const int st = n & 1, slot = n % SY_RAW;
        if (n >= 2) {
            sy_mbar_wait(sy_smem_u32(&s_bar[st]), ((n >> 1) - 1) & 1);     // the MMAs that read stage st (chunk n - 2) are complete
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            while ((gf + 1) * SY_FL - 1 <= n - 2) flush(gf++);
        }
        __syncwarp();                                    // this warp's copies of chunk n have landed; its weights are visible
        unsigned char* stage = sy_sm + (size_t)st * SY_STAGE_BYTES;
        const float* rawc = raw_warp + (size_t)slot * (SY_RAW_BYTES / 4) + lane;
#pragma unroll
        for (int oo = 0; oo < SY_KC / 16; ++oo) {
            const int o = og * (SY_KC / 16) + oo;
            float v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = rawc[(oo * 8 + k) * SY_T];
            if (side == 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    if (diag) dsum = fma((double)v[k], (double)s_wd[warp][slot][oo * 8 + k], dsum);
                    v[k] *= s_w[warp][slot][oo * 8 + k];
                }
            } else {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] *= sB;
            }
            uint4 hi, lo;
            sy_split(v, hi, lo);
            // K-step o / 2, K half o & 1
            if (side == 0) {
                const uint32_t off = (uint32_t)(o >> 1) * (2u * SY_T * 16u) + (uint32_t)(o & 1) * (SY_T * 16u) + row_off;
                *reinterpret_cast<uint4*>(stage + off) = hi;
                *reinterpret_cast<uint4*>(stage + SY_A_BYTES + off) = lo;
            } else {
                const uint32_t off = (uint32_t)(o >> 1) * (2u * 2u * SY_T * 16u) + (uint32_t)(o & 1) * (2u * SY_T * 16u) + row_off;
                *reinterpret_cast<uint4*>(stage + 2 * SY_A_BYTES + off) = hi;                    // rows 0..127: B1
                *reinterpret_cast<uint4*>(stage + 2 * SY_A_BYTES + SY_T * 16 + off) = lo;        // rows 128..255: B2
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        // only warp 0 waits for the chunk to be complete (named barrier 1 + st: 480 arrives + its own 32); the other warps go on
        // to the next chunk, held back by the "empty" mbarrier of their stage alone
        if (warp != 0) asm volatile("bar.arrive %0, %1;" ::"r"(1 + st), "r"(SY_THREADS) : "memory");
        else asm volatile("bar.sync %0, %1;" ::"r"(1 + st), "r"(SY_THREADS) : "memory");
        if (warp == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            if (sy_elect_one()) {
                const int g = n / SY_FL;
                const uint32_t d = tmem + (uint32_t)(g & 1) * 256u;
                uint32_t accum = (n - g * SY_FL) ? 1u : 0u;
                const uint32_t sa = sm_base + (uint32_t)st * SY_STAGE_BYTES;
                const uint32_t desc_hi = (128u >> 4) | (1u << 14);
                const uint32_t a1 = ((sa >> 4) & 0x3FFFu) | ((((uint32_t)(SY_T * 16) >> 4) & 0x3FFFu) << 16);
                const uint32_t a2 = (((sa + SY_A_BYTES) >> 4) & 0x3FFFu) | ((((uint32_t)(SY_T * 16) >> 4) & 0x3FFFu) << 16);
                const uint32_t bd = (((sa + 2 * SY_A_BYTES) >> 4) & 0x3FFFu) | ((((uint32_t)(2 * SY_T * 16) >> 4) & 0x3FFFu) << 16);
#pragma unroll
                for (int ks = 0; ks < SY_KC / 16; ++ks) {
                    const uint32_t astep = (uint32_t)((ks * 2 * SY_T * 16) >> 4), bstep = (uint32_t)((ks * 4 * SY_T * 16) >> 4);
                    sy_mma_lo(d, a1 + astep, bd + bstep, desc_hi, idesc256, accum);     // hi.hi | hi.lo
                    sy_mma_lo(d, a2 + astep, bd + bstep, desc_hi, idesc128, 1u);        // lo.hi into columns 0..127
                    accum = 1u;
                }
                sy_commit(sy_smem_u32(&s_bar[st]));
            }
            __syncwarp();
        }
    }
    asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    const int n = nrel;
    if (n > 0) {
        if (tid == 0) sy_commit(sy_smem_u32(&s_bar[2]));                   // arrives when every MMA issued so far is complete
        sy_mbar_wait(sy_smem_u32(&s_bar[2]), 0);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        while (gf * SY_FL < n) flush(gf++);
    }
    // epilogue: lower triangle of A = F + lambda g (fp64), D on diagonal tiles
    const double lam = lam_reg ? (double)lam_reg[b] : 0.0;
    double* Ab = A + (size_t)b * ns * ns;
    const int i = i0 + 32 * lq + lane;
    if (i < ns) {
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            const int j = j0 + cq * 32 + k;
            if (j <= i) Ab[(size_t)i * ns + j] = (double)(acc[k] * unscale) + lam * px_curv(i, j, nsx, nsy);
        }
    }
    if (diag) {
        if (side == 0) s_d[og * SY_T + c] = dsum;
        __syncthreads();
        if (tid < SY_T && i0 + tid < ns) Dv[(size_t)b * ns + i0 + tid] = s_d[tid] + s_d[SY_T + tid];
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512) : "memory");
}

cudaError_t launch_pixsrc_syrk_tc(glad_ctx* c, cudaStream_t st, const float* f, const int2* rng, const float* d_lam, int npix, int ns,
                                  int nsx, int nsy, int Bc, const double* stat, unsigned short* rowlist, double* A, double* D) {
    const size_t smem = 2 * (size_t)SY_STAGE_BYTES + SY_RAW * (size_t)SY_RAW_BYTES;
    cudaError_t e = smem_optin(c, pixsrc_syrk_tc_kernel);
    if (e != cudaSuccess) return e;
    const int nt = (ns + SY_T - 1) / SY_T;
    pixsrc_syrk_tc_kernel<<<dim3(nt * (nt + 1) / 2, Bc), SY_THREADS, smem, st>>>(f, c->d_ivar, c->d_data, rng, d_lam, stat, npix, ns, nsx, nsy, rowlist, A, D);
    return cudaGetLastError();
}
