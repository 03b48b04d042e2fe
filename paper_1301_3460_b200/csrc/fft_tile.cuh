// fft_tile.cuh -- in-place power-of-two FFTs along one axis of a shared-memory tile (fp64, sm_100a).
//
// Forward transforms are decimation-in-frequency: natural order in, DIGIT-REVERSED order out.  Inverse
// transforms are the exact stage-by-stage inverses (decimation-in-time, conjugate twiddles), so they take
// digit-reversed order in and give natural order out.  Between the two, the p2max/p2 filter is applied at
// the stored (digit-reversed) positions using per-axis tables built in the same order (host side,
// lgf_api.cu: stored_freq()).  No reordering pass and no ping-pong buffer is ever needed.
//
// Stage radices (the "plan" of an axis, AxisPlan) are fixed per axis by the host (lgf_api.cu make_plan):
//   "a" axes (0 and 2):  L = 4:[4]  8:[8]  16:[4,4]  32:[8,4]  64:[8,8]  128:[8,4,4]
//   "b" axes (1 and 3):  the same except 32:[4,8], so that the last a-stage and the first b-stage of a 32x32 or
//   16x16 tile are both radix 4 and can be fused into one 16-point register block (fft_fast.cuh).
// The last forward stage has unit twiddles.
#pragma once
#include "su3.cuh"

namespace lgf {

struct AxisPlan {
    int nst;       // number of stages
    int lgr[3];    // log2 radix of each forward stage, in forward order
};

// One axis transform inside a tile.  Work items are (iA, q, iB): iA the fastest thread index over a
// non-transformed tile axis (stride strideA, 2^lgA values), q the butterfly inside a line, iB the slow
// non-transformed axis.
struct AxisXf {
    int lgL;       // log2 of the transform length
    int strideK;   // element stride along the transformed axis
    int lgA, strideA;
    int nB, strideB;
    const cplx* tw;  // shared-memory table tw[k] = exp(-2 pi i k / L), k < L
    AxisPlan plan;
};

template <bool INV> __device__ __forceinline__ cplx mul_i(cplx a) {  // forward: * (-i); inverse: * (+i)
    return INV ? mk(-a.y, a.x) : mk(a.y, -a.x);
}

template <bool INV> __device__ __forceinline__ void bfly2(cplx& a, cplx& b) { cplx t = csub(a, b); a = cadd(a, b); b = t; }

// y_m = sum_k x_k W4^{mk}, W4 = exp(-+ 2 pi i/4)
template <bool INV> __device__ __forceinline__ void bfly4(cplx& x0, cplx& x1, cplx& x2, cplx& x3) {
    cplx t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), t3 = mul_i<INV>(csub(x1, x3));
    x0 = cadd(t0, t2); x2 = csub(t0, t2); x1 = cadd(t1, t3); x3 = csub(t1, t3);
}

template <bool INV> __device__ __forceinline__ void bfly8(cplx (&v)[8]) {
    // even/odd split: E = DFT4(v0,v2,v4,v6), O = DFT4(v1,v3,v5,v7); y_m = E_m + W8^m O_m, y_{m+4} = E_m - W8^m O_m
    bfly4<INV>(v[0], v[2], v[4], v[6]);   // now v0,v2,v4,v6 = E_0..E_3
    bfly4<INV>(v[1], v[3], v[5], v[7]);   // now v1,v3,v5,v7 = O_0..O_3
    const real h = (real)0.70710678118654752440;
    cplx o1 = v[3], o2 = v[5], o3 = v[7];
    // W8^1 = h(1 -+ i), W8^2 = -+ i, W8^3 = h(-1 -+ i)
    cplx w1 = INV ? mk(h * (o1.x - o1.y), h * (o1.x + o1.y)) : mk(h * (o1.x + o1.y), h * (o1.y - o1.x));
    cplx w2 = mul_i<INV>(o2);
    cplx w3 = INV ? mk(-h * (o3.x + o3.y), h * (o3.x - o3.y)) : mk(h * (o3.y - o3.x), -h * (o3.x + o3.y));
    cplx e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
    v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
    v[1] = cadd(e1, w1); v[5] = csub(e1, w1);
    v[2] = cadd(e2, w2); v[6] = csub(e2, w2);
    v[3] = cadd(e3, w3); v[7] = csub(e3, w3);
}

// 16 points as 4 x 4 in place, DIGIT-REVERSED frequency order: forward takes the points x_m (m = c + 4r) in v[m] and leaves
// F_k = sum_m x_m W16^{km}, k = q + 4p, in v[p + 4q]; the inverse is the exact mirror (frequencies in, points out).
// This is the order two successive radix-4 stages of the generic passes produce, so a radix-16 stage here and the
// plan [4,4] there store the same frequency at the same position.
template <bool INV> __device__ __forceinline__ cplx mul_w16(cplx a, int e) {      // a * W16^e (forward) or a * conj(W16^e); e = q c <= 9
    const real c1 = (real)0.92387953251128675613, s1 = (real)0.38268343236508977173, h = (real)0.70710678118654752440;
    // W16^e = (cos, -sin)(2 pi e / 16)
    real wr, wi;
    switch (e) {
        case 0: return a;
        case 1: wr = c1; wi = -s1; break;
        case 2: wr = h; wi = -h; break;
        case 3: wr = s1; wi = -c1; break;
        case 4: return mul_i<INV>(a);
        case 6: wr = -h; wi = -h; break;
        default: wr = -c1; wi = s1; break;      // 9
    }
    if (INV) wi = -wi;
    return mk(a.x * wr - a.y * wi, a.x * wi + a.y * wr);
}
template <bool INV> __device__ __forceinline__ void bfly16(cplx (&v)[16]) {
    if constexpr (!INV) {
#pragma unroll
        for (int c = 0; c < 4; c++) bfly4<false>(v[c], v[c + 4], v[c + 8], v[c + 12]);      // over r: t[c][q] in v[c + 4q]
#pragma unroll
        for (int q = 1; q < 4; q++)
#pragma unroll
            for (int c = 1; c < 4; c++) v[c + 4 * q] = mul_w16<false>(v[c + 4 * q], q * c);
#pragma unroll
        for (int q = 0; q < 4; q++) bfly4<false>(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);   // over c: F_{q+4p} in v[p + 4q]
    } else {
#pragma unroll
        for (int q = 0; q < 4; q++) bfly4<true>(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
#pragma unroll
        for (int q = 1; q < 4; q++)
#pragma unroll
            for (int c = 1; c < 4; c++) v[c + 4 * q] = mul_w16<true>(v[c + 4 * q], q * c);
#pragma unroll
        for (int c = 0; c < 4; c++) bfly4<true>(v[c], v[c + 4], v[c + 8], v[c + 12]);
    }
}
// frequency digit held in slot s of a radix-R butterfly's output (input of the inverse)
template <int R> __host__ __device__ constexpr int slot_freq(int s) { return (R == 16) ? ((s >> 2) + 4 * (s & 3)) : s; }

template <int R, bool INV> __device__ __forceinline__ void bfly(cplx (&v)[R]) {
    if constexpr (R == 2) bfly2<INV>(v[0], v[1]);
    if constexpr (R == 4) bfly4<INV>(v[0], v[1], v[2], v[3]);
    if constexpr (R == 8) bfly8<INV>(v);
    if constexpr (R == 16) bfly16<INV>(v);
}

// One radix-R stage on sub-blocks of length N = 2^lgN for every line of the tile.  The caller syncs.
template <int R, bool INV>
__device__ __forceinline__ void fft_stage(cplx* __restrict__ t, const AxisXf& a, int lgN) {
    constexpr int lgR = (R == 8) ? 3 : (R == 4 ? 2 : 1);
    const int lgs = lgN - lgR;            // s = N/R: stride between the R inputs of one butterfly
    const int lgQ = a.lgL - lgR;          // butterflies per line
    const int nwork = a.nB << (a.lgA + lgQ);
    const int twsh = a.lgL - lgN;         // W_N^k = tw[k << twsh]
    const int ss = a.strideK << lgs;
    for (int w = threadIdx.x; w < nwork; w += blockDim.x) {
        const int iA = w & ((1 << a.lgA) - 1);
        const int q = (w >> a.lgA) & ((1 << lgQ) - 1);
        const int iB = w >> (a.lgA + lgQ);
        const int j = q & ((1 << lgs) - 1);
        const int b = q >> lgs;
        cplx* p = t + iA * a.strideA + iB * a.strideB + ((b << lgN) + j) * a.strideK;
        cplx v[R];
#pragma unroll
        for (int m = 0; m < R; m++) v[m] = p[m * ss];
        if (INV) {
            if (lgs > 0) {
#pragma unroll
                for (int m = 1; m < R; m++) v[m] = cmulc(v[m], a.tw[(j * m) << twsh]);
            }
            bfly<R, true>(v);
        } else {
            bfly<R, false>(v);
            if (lgs > 0) {
#pragma unroll
                for (int m = 1; m < R; m++) v[m] = cmul(v[m], a.tw[(j * m) << twsh]);
            }
        }
#pragma unroll
        for (int m = 0; m < R; m++) p[m * ss] = v[m];
    }
}

template <bool INV> __device__ __forceinline__ void fft_stage_dispatch(cplx* t, const AxisXf& a, int lgN, int lgR) {
    if (lgR == 3) fft_stage<8, INV>(t, a, lgN);
    else if (lgR == 2) fft_stage<4, INV>(t, a, lgN);
    else fft_stage<2, INV>(t, a, lgN);
}

// Forward (DIF) transform of every line along the axis; ends with __syncthreads().
__device__ __forceinline__ void fft_axis_forward(cplx* t, const AxisXf& a) {
    int lgN = a.lgL;
    for (int k = 0; k < a.plan.nst; k++) {
        fft_stage_dispatch<false>(t, a, lgN, a.plan.lgr[k]);
        __syncthreads();
        lgN -= a.plan.lgr[k];
    }
}
// Inverse (DIT) transform: the forward stages undone in reverse order; ends with __syncthreads().
__device__ __forceinline__ void fft_axis_inverse(cplx* t, const AxisXf& a) {
    int lgN = 0;
    for (int k = a.plan.nst - 1; k >= 0; k--) {
        lgN += a.plan.lgr[k];
        fft_stage_dispatch<true>(t, a, lgN, a.plan.lgr[k]);
        __syncthreads();
    }
}

}  // namespace lgf
