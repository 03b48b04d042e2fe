// fused_update.cuh -- S3/S4 of iteration k fused with S1 and FFT pass A of iteration k+1 (fp64, sm_100a).
//
// The separate passes read every link three times per iteration (S1, S4) and write it once.  The new links exist in
// registers at the end of S4, and Delta of the next iteration is LINEAR in them,
//     A(x) = sum_mu [U_mu(x-mu) - U_mu(x)],  Delta = (A - A^dag) - (1/3) Tr(A - A^dag)              [north_star step 1]
// so one kernel can do   U' = g U g^dag(x+mu)  ->  Delta'(x)  ->  theta', F' partials  ->  forward FFT over axes 0,1
// and the links cross HBM twice per iteration (one read, one write) instead of three times.
//
// One CTA per (x2,x3) plane, as in pass A.  A warp walks its rows of the plane in order; per site a thread
//   * rotates its four links (S4) and stores them,
//   * subtracts their packed contributions c_mu(x) from Delta'(x),
//   * adds the backward contributions: c_0(x-0) from the neighbouring lane (shuffle), c_1(x-1) from its own previous
//     row (registers), and c_2(x-2), c_3(x-3) -- links owned by other CTAs -- by rotating those two links again.
// The first row of a warp's range gets c_1 from the last row of another warp: both sides add into a zeroed tile
// entry with shared-memory atomics; an entry receives exactly two addends, so the sum does not depend on their order.
// Because other CTAs still read the old U_2(x-2), U_3(x-3) while this one writes, the links are double-buffered:
// read from buffer ctl->parity, write to the other; k_finalize flips the parity.
// g(x) comes from gbuf (rows 0,1 stored by pass C, k_fa_inv<..., WRITE_G>).
#pragma once
#include "fft_fast.cuh"

#ifndef LGF_FU_NT
#define LGF_FU_NT 128
#endif
#ifndef LGF_FU_MINB
#define LGF_FU_MINB 3
#endif
// L2 bulk-prefetch distance in warp iterations (0 = off).  Measured on B200 at 32^4: 282.7 us off, 325.8 us at 2,
// 331.7 us at 4 -- the kernel is bound by SM<->L2 traffic, not by DRAM latency, so prefetching only adds contention.
#ifndef LGF_FU_PFD
#define LGF_FU_PFD 0
#endif

namespace lgf {

// Packed contribution of one link W to Delta:  (W - W^dag) - (1/3) Tr(W - W^dag), components (01, 02, 12, (Im 00, Im 11)).
__device__ __forceinline__ void link_contrib(const cplx (&w)[9], cplx (&c)[4]) {
    c[0] = mk(w[1].x - w[3].x, w[1].y + w[3].y);
    c[1] = mk(w[2].x - w[6].x, w[2].y + w[6].y);
    c[2] = mk(w[5].x - w[7].x, w[5].y + w[7].y);
    const double tr3 = (2.0 / 3.0) * (w[0].y + w[4].y + w[8].y);
    c[3] = mk(2.0 * w[0].y - tr3, 2.0 * w[4].y - tr3);
}
// Tr[Delta Delta^dag] of a packed Delta
__device__ __forceinline__ double packed_norm(const cplx (&a)[4]) {
    const double e2 = a[3].x + a[3].y;
    return 2.0 * (cnorm2(a[0]) + cnorm2(a[1]) + cnorm2(a[2])) + a[3].x * a[3].x + a[3].y * a[3].y + e2 * e2;
}
__device__ __forceinline__ void load_g(const cplx* __restrict__ gbuf, long long V, long long x, cplx (&g)[9]) {
#pragma unroll
    for (int c = 0; c < 6; c++) g[c] = ldg2(gbuf + (long long)c * V + x);
}
__device__ __forceinline__ cplx shfl_c(cplx v, int src, int width) {
    return mk(__shfl_sync(0xffffffffu, v.x, src, width), __shfl_sync(0xffffffffu, v.y, src, width));
}

template <int LG0, int LG1, int NC, int NT>
__global__ void __launch_bounds__(NT, LGF_FU_MINB) k_fu_update_delta_fwd(cplx* __restrict__ links2, long long buf_stride, const cplx* __restrict__ gbuf,
                                                                         cplx* __restrict__ field, double2* __restrict__ partials, Geom G, FftTables T,
                                                                         const Ctl* __restrict__ ctl) {
    pdl_enter();
    if (ctl->done) return;
    using PA = Plan2<LG0, false>;
    using PB = Plan2<LG1, true>;
    constexpr int L0 = PA::L, L1 = PB::L, S = L0 + 1, SC = S * L1, nP = L0 * L1;
    constexpr int NW = NT / 32, SPW = nP / NW, NIT = SPW / 32;
    constexpr int NR = (NC == 6) ? 2 : 3;
    static_assert(LG0 <= 5, "a row must fit in a warp");
    static_assert(SPW % 32 == 0 && SPW % L0 == 0 && NIT >= 1, "a warp covers whole rows");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw0 = tile + 4 * SC;
    cplx* tw1 = tw0 + L0;
    __shared__ double red[64];

    const long long V = G.V;
    const int par = ctl->parity;
    const cplx* __restrict__ lin = links2 + (long long)par * buf_stride;
    cplx* __restrict__ lout = links2 + (long long)(par ^ 1) * buf_stride;

    const int plane = blockIdx.x, L2 = G.L[2], L3 = G.L[3];
    const int x2 = plane & (L2 - 1), x3 = plane >> G.lg[2];
    auto pbase = [&](int a2, int a3) { return (long long)((a2 & (L2 - 1)) + ((a3 & (L3 - 1)) << G.lg[2])) << (LG0 + LG1); };
    const long long xbase = pbase(x2, x3);
    const long long xb_f2 = pbase(x2 + 1, x3), xb_b2 = pbase(x2 - 1, x3), xb_f3 = pbase(x2, x3 + 1), xb_b3 = pbase(x2, x3 - 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // DRAM -> L2 prefetch of the 32 sites of warp iteration `it2`: one 512 B run per link entry and per g entry
    auto prefetch_it = [&](int it2) {
        if (LGF_FU_PFD > 0 && it2 < NIT) {
            const long long e0 = xbase + warp * SPW + it2 * 32;
            if (lane < 4 * NC) prefetch_l2(lin + (long long)lane * V + e0, 512);
            if (4 * NC > 32 && lane + 32 < 4 * NC) prefetch_l2(lin + (long long)(lane + 32) * V + e0, 512);
            if (lane < 6) prefetch_l2(gbuf + (long long)lane * V + e0, 512);
        }
    };
#pragma unroll
    for (int d = 0; d < LGF_FU_PFD; d++) prefetch_it(d);

    for (int i = threadIdx.x; i < L0; i += NT) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += NT) tw1[i] = T.tw[1][i];
    // the first row of every warp's range receives two atomic addends: zero it
    for (int i = threadIdx.x; i < 4 * NW * L0; i += NT) {
        const int c = i / (NW * L0), r = i % (NW * L0);
        const int e = (r / L0) * SPW + (r % L0);
        tile[c * SC + (e & (L0 - 1)) + (e >> LG0) * S] = mk(0.0, 0.0);
    }
    __syncthreads();

    double th = 0, fs = 0;
    cplx c1prev[4];
#pragma unroll
    for (int k = 0; k < 4; k++) c1prev[k] = mk(0.0, 0.0);

#pragma unroll 1
    for (int it = 0; it < NIT; it++) {
        prefetch_it(it + LGF_FU_PFD);
        const int e = warp * SPW + it * 32 + lane;
        const int x0 = e & (L0 - 1), x1 = e >> LG0;
        const long long x = xbase + e;
        cplx g[9];
        load_g(gbuf, V, x, g);
        third_row(g);
        cplx acc[4], c0[4], c1[4];
#pragma unroll
        for (int k = 0; k < 4; k++) acc[k] = mk(0.0, 0.0);
        // S4 for the four links of x, and their contributions -c_mu(x)
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            long long xf;
            if (mu == 0) xf = xbase + (e & ~(L0 - 1)) + ((x0 + 1) & (L0 - 1));
            else if (mu == 1) xf = xbase + (((x1 + 1) & (L1 - 1)) << LG0) + x0;
            else if (mu == 2) xf = xb_f2 + e;
            else xf = xb_f3 + e;
            cplx gp[9], u[9], w[9];
            load_g(gbuf, V, xf, gp);
            third_row(gp);
            load_link<NC>(lin, V, mu, x, u);
            rotate_link<NR>(g, u, gp, w);
            store_link<NC>(lout, V, mu, x, w);
            if (NC == 6) third_row(w);
            fs += w[0].x + w[4].x + w[8].x;
            cplx c[4];
            link_contrib(w, c);
#pragma unroll
            for (int k = 0; k < 4; k++) acc[k] = csub(acc[k], c[k]);
            if (mu == 0) {
#pragma unroll
                for (int k = 0; k < 4; k++) c0[k] = c[k];
            }
            if (mu == 1) {
#pragma unroll
                for (int k = 0; k < 4; k++) c1[k] = c[k];
            }
        }
        // +c_2(x-2), +c_3(x-3): links of other planes, rotated again here
#pragma unroll
        for (int mu = 2; mu < 4; mu++) {
            const long long xb = (mu == 2 ? xb_b2 : xb_b3) + e;
            cplx gm[9], u[9], w[9];
            load_g(gbuf, V, xb, gm);
            if (NC == 9) third_row(gm);
            load_link<NC>(lin, V, mu, xb, u);
            rotate_link<NR>(gm, u, g, w);
            if (NC == 6) third_row(w);
            cplx c[4];
            link_contrib(w, c);
#pragma unroll
            for (int k = 0; k < 4; k++) acc[k] = cadd(acc[k], c[k]);
        }
        // +c_0(x-0): the lane to the left in the same row
#pragma unroll
        for (int k = 0; k < 4; k++) acc[k] = cadd(acc[k], shfl_c(c0[k], (lane - 1) & (L0 - 1), L0));
        // +c_1(x-1): the row below -- this lane's previous iteration (L0 = 32), or the other half-warp (L0 = 16)
#pragma unroll
        for (int k = 0; k < 4; k++) {
            cplx b;
            if constexpr (L0 == 32) b = c1prev[k];
            else b = shfl_c((lane < 32 - L0) ? c1[k] : c1prev[k], (lane - L0) & 31, 32);
            acc[k] = cadd(acc[k], b);
            c1prev[k] = c1[k];
        }
        cplx* tp = tile + x0 + x1 * S;
        if (it == 0 && lane < L0) {          // c_1(x-1) comes from another warp: both add into the zeroed entry
#pragma unroll
            for (int k = 0; k < 4; k++) {
                double* q = reinterpret_cast<double*>(tp + k * SC);
                atomicAdd(q, acc[k].x); atomicAdd(q + 1, acc[k].y);
            }
        } else {
#pragma unroll
            for (int k = 0; k < 4; k++) tp[k * SC] = acc[k];
            th += packed_norm(acc);
        }
        if (it == NIT - 1 && lane >= 32 - L0) {   // last row of this warp's range: its c_1 belongs to the next warp's first row
            double* q = reinterpret_cast<double*>(tile + x0 + ((x1 + 1) & (L1 - 1)) * S);
#pragma unroll
            for (int k = 0; k < 4; k++) { atomicAdd(q + 2 * k * SC, c1[k].x); atomicAdd(q + 2 * k * SC + 1, c1[k].y); }
        }
    }
    __syncthreads();
    if (lane < L0) {                          // theta of the first rows, complete now
        const int e = warp * SPW + lane;
        const cplx* tp = tile + (e & (L0 - 1)) + (e >> LG0) * S;
        cplx a[4];
#pragma unroll
        for (int k = 0; k < 4; k++) a[k] = tp[k * SC];
        th += packed_norm(a);
    }
    block_sum2(th, fs, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(th, fs);
    __syncthreads();

    plane_forward_store<LG0, LG1, NT>(tile, tw0, tw1, field, V, xbase, Grp{(int)threadIdx.x, 0});
}

}  // namespace lgf
