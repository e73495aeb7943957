// Batched Cholesky factorisation A = L L^T (fp64, lower triangle in place) of the B matrices F + lambda g of the pixelated-source
// likelihood (Eq. 40, 43), N_s = 100 .. 4096.  Right-looking, panel width 64, THREE kernels per panel over the whole
// batch instead of one CTA per matrix:
//   chol_diag_kernel    CTA per matrix: the 64 x 64 diagonal block in shared memory; ln det and the not-positive-definite flag
//                       and W = L11^-1
//   chol_trsm_kernel    CTA per (64 rows below the block, matrix): L21 = A21 W^T as a 64 x 64 x 64 tile product (DMMA)
//   chol_update_kernel  CTA per (row of 64 x 64 tiles of the trailing lower triangle, matrix): A22 -= L21 L21^T on the fp64
//                       tensor-core path (DMMA m8n8k4), the panel tiles streamed through shared memory by cp.async
// The version this replaces ran the whole factorisation in one CTA per matrix (profiles/r1e.md: fp64 pipe 20 % active, 12 TFLOP/s,
// and at the paper's 64 x 64 source grid only 54 matrices fit the scratch, so 54 CTAs on 148 SMs: 2.47 s per 296 matrices).
// Here every trailing update is a grid of (tiles x matrices) CTAs whatever the batch size.
#include <math.h>

#include "glad_internal.h"

#define CH_NB 64
#define CH_P 65            // pitch (doubles) of the shared-memory tiles
#define CH_OUT 6           // doubles per vector in `out` (pixsrc_kernels.cu PX_OUT): [0] ln det A, [3] not-positive-definite flag

// D (8 x 8) = A (8 x 4, row-major) B (4 x 8, column-major) + C on the fp64 tensor-core path: a thread holds A[lane/4][lane%4],
// B[lane%4][lane/4] and C[lane/4][2 (lane%4) + {0, 1}]
__device__ __forceinline__ void ch_dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

#define CH_PU 68           // pitch (doubles) of the update kernel's tiles: 2 * 68 mod 32 = 8, so the 16 lanes of a half-warp
                           // (4 rows x 4 consecutive k) read 16 different bank pairs


__global__ void __launch_bounds__(256) chol_diag_kernel(double* __restrict__ A, int ns, int k0, double* __restrict__ out,
                                                        double* __restrict__ Winv) {
    __shared__ double L[CH_NB * CH_P];
    __shared__ double s_ld, s_isq[CH_NB], s_lg[CH_NB];
    __shared__ int s_bad;
    const int b = blockIdx.x, tid = threadIdx.x;
    double* Ab = A + (size_t)b * ns * ns;
    const int nb = min(CH_NB, ns - k0);
    if (tid == 0) { s_ld = 0.0; s_bad = 0; }
    for (int e = tid; e < CH_NB * CH_NB; e += 256) {
        const int r = e >> 6, c = e & 63;
        L[r * CH_P + c] = (r < nb && c <= r) ? Ab[(size_t)(k0 + r) * ns + k0 + c] : (r == c ? 1.0 : 0.0);
    }
    __syncthreads();
    // Elimination with UNSCALED columns and one barrier per step: column j and the pivot d_j = L[j][j] are final after step j - 1
    // and are not written again, so step j reads them and updates the trailing lower triangle with L[r][j] L[c][j] / d_j; the
    // scaling L[r][j] /= sqrt(d_j) of every column, the square roots and the logarithms wait until the elimination is over.  (Pivot,
    // barrier, column scaling, barrier, update, barrier per step: the barriers and thread 0's sqrt / log were most of the kernel.)
    // Thread (tr, tc) of a 16 x 16 arrangement takes rows j+1+tr, +16, .. and columns j+1+tc, +16, .. <= row.
    {
        const int tr = tid >> 4, tc = tid & 15;
        for (int j = 0; j < nb; ++j) {
            const double d = L[j * CH_P + j];
            const bool okd = (d > 0.0) && isfinite(d);
            const double invd = okd ? 1.0 / d : 1.0;               // a pivot that is not positive is flagged and taken as 1
            for (int r = j + 1 + tr; r < nb; r += 16) {
                const double lrj = L[r * CH_P + j] * invd;
                for (int c = j + 1 + tc; c <= r; c += 16) L[r * CH_P + c] = fma(-lrj, L[c * CH_P + j], L[r * CH_P + c]);
            }
            __syncthreads();
        }
    }
    if (tid < nb) {                                                // thread j: pivot j -> ln det, flag, 1 / sqrt(d_j)
        const double d = L[tid * CH_P + tid];
        const bool okd = (d > 0.0) && isfinite(d);
        if (!okd) s_bad = 1;
        s_isq[tid] = okd ? rsqrt(d) : 1.0;
        s_lg[tid] = okd ? log(d) : 0.0;
    }
    __syncthreads();
    for (int e = tid; e < CH_NB * CH_NB; e += 256) {
        const int r = e >> 6, c = e & 63;
        if (r < nb && c <= r) {                                     // (only thread (c, c) touches the pivot itself)
            const double v = L[r * CH_P + c];
            L[r * CH_P + c] = (r == c) ? (((v > 0.0) && isfinite(v)) ? sqrt(v) : 1.0) : v * s_isq[c];
        }
    }
    if (tid == 0) { double t = 0.0; for (int j = 0; j < nb; ++j) t += s_lg[j]; s_ld = t; }
    __syncthreads();
    for (int e = tid; e < CH_NB * CH_NB; e += 256) {
        const int r = e >> 6, c = e & 63;
        if (r < nb && c <= r) Ab[(size_t)(k0 + r) * ns + k0 + c] = L[r * CH_P + c];
    }
    if (tid == 0) {
        double* o = out + (size_t)b * CH_OUT;
        o[0] = (k0 == 0 ? 0.0 : o[0]) + s_ld;
        o[3] = (k0 == 0 ? 0.0 : o[3]) + (s_bad ? 1.0 : 0.0);
    }
    // W = L11^-1 for the panel kernel (only full blocks have rows below them): thread c solves L11 x = e_c by forward substitution
    if (nb == CH_NB && k0 + CH_NB < ns && tid < CH_NB) {
        // column-oriented: once x[r] is known, the 63 - r updates v[r'] -= L[r'][r] x[r] are independent of one another (the
        // row-oriented form is one chain of 2016 dependent DFMAs per thread: half of this kernel's 184 us)
        double* Wb = Winv + (size_t)b * CH_NB * CH_NB;
        double v[CH_NB];
#pragma unroll
        for (int r = 0; r < CH_NB; ++r) v[r] = (r == tid) ? 1.0 : 0.0;
#pragma unroll
        for (int r = 0; r < CH_NB; ++r) {
            v[r] = v[r] / L[r * CH_P + r];
#pragma unroll
            for (int k = r + 1; k < CH_NB; ++k) v[k] = fma(-L[k * CH_P + r], v[r], v[k]);
        }
#pragma unroll
        for (int r = 0; r < CH_NB; ++r) Wb[r * CH_NB + tid] = v[r];     // W[r][c]
    }
}

// L21 = A21 L11^-T = A21 W^T with W = L11^-1 from chol_diag_kernel: a 64-row tile of the panel times a 64 x 64 matrix, the same
// sum_k P_i[i,k] P_j[c,k] form as the trailing update and, like it, on the DMMA path (a thread per row with its 64 doubles in
// registers took 3.2 of 15 ms; 4 x 4 doubles per thread with DFMA 1.7 of 10.6)
__global__ void __launch_bounds__(256, 2) chol_trsm_kernel(double* __restrict__ A, const double* __restrict__ Winv, int ns, int k0) {
    extern __shared__ double ch_sm[];
    double* Pi = ch_sm;                     // [row of the tile][k], pitch CH_PU
    double* Pj = ch_sm + CH_NB * CH_PU;     // [c][k] = W[c][k]
    const int b = blockIdx.y, tid = threadIdx.x;
    const int ib = k0 + CH_NB + blockIdx.x * CH_NB;
    double* Ab = A + (size_t)b * ns * ns;
    const double* Wb = Winv + (size_t)b * CH_NB * CH_NB;
    for (int e = tid; e < CH_NB * CH_NB; e += 256) {
        const int r = e >> 6, k = e & 63;
        Pi[r * CH_PU + k] = (ib + r < ns) ? Ab[(size_t)(ib + r) * ns + k0 + k] : 0.0;
        Pj[r * CH_PU + k] = Wb[r * CH_NB + k];
    }
    __syncthreads();
    const int warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    const int wr = (warp >> 1) * 16, wc = (warp & 1) * 32;      // the warp's 16 rows and 32 columns of the tile
    const double* pa = Pi + (wr + g) * CH_PU + q;
    const double* pb = Pj + (wc + g) * CH_PU + q;
    double acc[2][4][2];
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
        for (int n = 0; n < 4; ++n) acc[m][n][0] = acc[m][n][1] = 0.0;
#pragma unroll 4
    for (int k = 0; k < CH_NB; k += 4) {
        double ar[2], br[4];
#pragma unroll
        for (int m = 0; m < 2; ++m) ar[m] = pa[m * 8 * CH_PU + k];
#pragma unroll
        for (int n = 0; n < 4; ++n) br[n] = pb[n * 8 * CH_PU + k];
#pragma unroll
        for (int m = 0; m < 2; ++m)
#pragma unroll
            for (int n = 0; n < 4; ++n) ch_dmma(acc[m][n][0], acc[m][n][1], ar[m], br[n]);
    }
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
        for (int n = 0; n < 4; ++n)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int i = ib + wr + 8 * m + g;
                if (i < ns) Ab[(size_t)i * ns + k0 + wc + 8 * n + 2 * q + e] = acc[m][n][e];
            }
}

__device__ __forceinline__ void ch_cp_async8(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(sa), "l"(gmem) : "memory");
}

// A[i, j] -= sum_k L21[i, k] L21[j, k] on the trailing lower triangle (rows / columns >= r0).  CTA = (row of 64 x 64 tiles ti, matrix):
// the panel rows of ti stay in shared memory, those of tj = 0 .. ti stream through a double buffer filled by cp.async one tile
// ahead (row-major [row][k]: 8-byte copies), and the A tile is fetched into registers before the tile product.  The product runs
// as DMMA m8n8k4 (warp = 16 x 32 outputs = 2 x 4 fragments: 6 shared-memory loads per 8 DMMAs = 64 multiply-adds per thread; the
// 4 x 4 DFMA form it replaces needed 8 loads per 16 and stopped at 45 % of the fp64 pipe: profiles/r2.md).  Rows of tiles are
// handed out longest first.
__device__ __forceinline__ void ch_cp_async16(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gmem) : "memory");
}

// EVEN: n_s is even, so every row of A starts on a 16-byte boundary and pairs of columns move as one 16-byte access
template <bool EVEN>
__global__ void __launch_bounds__(256, 2) chol_update_kernel(double* __restrict__ A, int ns, int k0, int nt) {
    extern __shared__ double ch_sm[];
    double* Pi = ch_sm;
    double* Pj = ch_sm + CH_NB * CH_PU;     // two buffers
    const int b = blockIdx.y, tid = threadIdx.x;
    const int ti = nt - 1 - (int)blockIdx.x;
    const int r0 = k0 + CH_NB, ib = r0 + ti * CH_NB;
    double* Ab = A + (size_t)b * ns * ns;
    auto fill = [&](double* dst, int rb) {         // rows rb .. rb + 63, columns k0 .. k0 + 63 of the panel
        if (EVEN) {
#pragma unroll
            for (int it = 0; it < (CH_NB * CH_NB) / 512; ++it) {
                const int e = tid + it * 256, r = e >> 5, k = (e & 31) * 2;
                if (rb + r < ns) ch_cp_async16(dst + r * CH_PU + k, Ab + (size_t)(rb + r) * ns + k0 + k);
                else { dst[r * CH_PU + k] = 0.0; dst[r * CH_PU + k + 1] = 0.0; }
            }
        } else {
#pragma unroll
            for (int it = 0; it < (CH_NB * CH_NB) / 256; ++it) {
                const int e = tid + it * 256, r = e >> 6, k = e & 63;
                if (rb + r < ns) ch_cp_async8(dst + r * CH_PU + k, Ab + (size_t)(rb + r) * ns + k0 + k);
                else dst[r * CH_PU + k] = 0.0;
            }
        }
        asm volatile("cp.async.commit_group;\n" ::: "memory");
    };
    fill(Pi, ib);
    fill(Pj, r0);
    const int warp = tid >> 5, lane = tid & 31, g = lane >> 2, q = lane & 3;
    const int wr = (warp >> 1) * 16, wc = (warp & 1) * 32;      // the warp's 16 rows and 32 columns of the tile
    const double* pa = Pi + (wr + g) * CH_PU + q;
    for (int tj = 0; tj <= ti; ++tj) {
        const int jb = r0 + tj * CH_NB;
        const double* Pc = Pj + (tj & 1) * CH_NB * CH_PU;
        if (tj < ti) fill(Pj + ((tj + 1) & 1) * CH_NB * CH_PU, jb + CH_NB);
        double cur[2][4][2], acc[2][4][2];
#pragma unroll
        for (int m = 0; m < 2; ++m)
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                const int i = ib + wr + 8 * m + g, j = jb + wc + 8 * n + 2 * q;
                if (EVEN) {                 // j is even and j <= i < n_s: j + 1 < n_s too, the pair is inside the row
                    const double2 v = (i < ns && j <= i) ? *reinterpret_cast<const double2*>(Ab + (size_t)i * ns + j) : make_double2(0.0, 0.0);
                    cur[m][n][0] = v.x; cur[m][n][1] = v.y;
                } else {
#pragma unroll
                    for (int e = 0; e < 2; ++e) cur[m][n][e] = (i < ns && j + e <= i) ? Ab[(size_t)i * ns + j + e] : 0.0;
                }
                acc[m][n][0] = acc[m][n][1] = 0.0;
            }
        if (tj < ti) asm volatile("cp.async.wait_group 1;\n" ::: "memory");
        else asm volatile("cp.async.wait_group 0;\n" ::: "memory");
        __syncthreads();
        const double* pb = Pc + (wc + g) * CH_PU + q;
#pragma unroll 4
        for (int k = 0; k < CH_NB; k += 4) {
            double ar[2], br[4];
#pragma unroll
            for (int m = 0; m < 2; ++m) ar[m] = pa[m * 8 * CH_PU + k];
#pragma unroll
            for (int n = 0; n < 4; ++n) br[n] = pb[n * 8 * CH_PU + k];
#pragma unroll
            for (int m = 0; m < 2; ++m)
#pragma unroll
                for (int n = 0; n < 4; ++n) ch_dmma(acc[m][n][0], acc[m][n][1], ar[m], br[n]);
        }
#pragma unroll
        for (int m = 0; m < 2; ++m)
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                const int i = ib + wr + 8 * m + g, j = jb + wc + 8 * n + 2 * q;
                if (EVEN && i < ns && j + 1 <= i)        // both below or on the diagonal: one 16-byte store
                    *reinterpret_cast<double2*>(Ab + (size_t)i * ns + j) = make_double2(cur[m][n][0] - acc[m][n][0], cur[m][n][1] - acc[m][n][1]);
                else {
#pragma unroll
                    for (int e = 0; e < 2; ++e)
                        if (i < ns && j + e <= i) Ab[(size_t)i * ns + j + e] = cur[m][n][e] - acc[m][n][e];
                }
            }
        __syncthreads();                   // the buffer just read is refilled by the next iteration's prefetch
    }
}

// the whole factorisation of Bc matrices on stream st; out[b*6 + 0] = ln det A, out[b*6 + 3] != 0 = not positive definite
size_t pixsrc_factor_scratch_bytes(int Bc) { return sizeof(double) * (size_t)Bc * CH_NB * CH_NB; }

// Winv: scratch of pixsrc_factor_scratch_bytes(Bc)
cudaError_t launch_pixsrc_factor(glad_ctx* c, cudaStream_t st, double* A, int ns, int Bc, double* out, double* Winv) {
    const size_t sm_trsm = sizeof(double) * 2 * CH_NB * CH_PU, sm_upd = sizeof(double) * 3 * CH_NB * CH_PU;
    cudaError_t e = smem_optin(c, chol_update_kernel<true>);
    if (e == cudaSuccess) e = smem_optin(c, chol_update_kernel<false>);
    if (e == cudaSuccess) e = smem_optin(c, chol_trsm_kernel);
    if (e != cudaSuccess) return e;
    for (int k0 = 0; k0 < ns; k0 += CH_NB) {
        chol_diag_kernel<<<Bc, 256, 0, st>>>(A, ns, k0, out, Winv);
        c->launches++;
        const int rest = ns - k0 - CH_NB;
        if (rest <= 0) break;
        const int nt = (rest + CH_NB - 1) / CH_NB;
        chol_trsm_kernel<<<dim3(nt, Bc), 256, sm_trsm, st>>>(A, Winv, ns, k0);
        if (ns % 2 == 0) chol_update_kernel<true><<<dim3(nt, Bc), 256, sm_upd, st>>>(A, ns, k0, nt);
        else chol_update_kernel<false><<<dim3(nt, Bc), 256, sm_upd, st>>>(A, ns, k0, nt);
        c->launches += 2;
    }
    return cudaGetLastError();
}
