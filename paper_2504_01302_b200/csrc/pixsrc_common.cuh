// Shared by the pixelated-source kernels (pixsrc_kernels.cu, pixsrc_syrk_tc.cu): the curvature regulariser's matrix g (R-P3).
#pragma once

// (T^2)[i, i'] of the (1,-2,1) second-difference matrix T with zeros outside, n points (R-P3)
__device__ __forceinline__ double px_t2(int i, int ip, int n) {
    const int d = i > ip ? i - ip : ip - i;
    if (d == 0) return 4.0 + (i > 0 ? 1.0 : 0.0) + (i < n - 1 ? 1.0 : 0.0);
    if (d == 1) return -4.0;
    if (d == 2) return 1.0;
    return 0.0;
}
__device__ __forceinline__ double px_curv(int a, int c, int nsx, int nsy) {
    const int ja = a / nsx, ia = a - ja * nsx, jc = c / nsx, ic = c - jc * nsx;
    double v = 0.0;
    if (ja == jc) v += px_t2(ia, ic, nsx);
    if (ia == ic) v += px_t2(ja, jc, nsy);
    return v;
}

