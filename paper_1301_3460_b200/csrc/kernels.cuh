// kernels.cuh -- the sm_100a kernels of one Fourier-accelerated gauge-fixing iteration (fp64).
//
// Data in HBM:
//   links  structure-of-arrays: entry c (0..NC-1; NC = 6 two-row / 9 full) of direction mu is one contiguous
//          V-array of double2 at links + (mu*NC + c)*V, site index x0 fastest  -> every warp load is 512 B
//          contiguous.
//   field  4 packed complex components of the traceless anti-Hermitian Delta / X:
//          f0 = M01, f1 = M02, f2 = M12, f3 = (Im M00, Im M11); component c at field + c*V.
//   gbuf   (optional) g(x) rows 0,1: 6 V-arrays of double2.
//
// Kernels:
//   k_delta        S1: Delta + block partials of theta, F                       (unfused variant)
//   k_fft01<MODE>  S2a/S2c on the (x0,x1) plane of one (x2,x3): forward or inverse 2-D FFT in shared memory;
//                  MODE_DELTA_FWD computes Delta of the plane itself (S1 fused), MODE_INV_G writes g (S3 fused)
//   k_fft23_mid    S2a+S2b+S2c on axes 2,3 for a chunk of x0: forward, p2max/p2 filter, inverse
//   k_finalize     deterministic final reduction of the partials, S5 stop flag
//   k_update_quad  S3+S4: rebuild g(x+mu) from X, one thread per link, rotate the link in place (default)
//   k_update_g     S3+S4 with g read from gbuf (LGF_OPT_STORE_G)
//   k_layout_in/out, k_plaquette, k_unpack_field, k_copy: boundary helpers
// The compile-time-sized passes live in fft_fast.cuh, their TMA-fed persistent forms (the default path) in fft_tma.cuh,
// the kernels of the slab-decomposed context in slab.cuh.
#pragma once
#include "su3.cuh"
#include "fft_tile.cuh"

namespace lgf {

// ------------------------------------------------------------------------------------------------ reductions
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// Block-wide sum of two values in a fixed order (warp shuffle tree, then warp 0 over the warp partials).
// Result valid in thread 0.  red must hold 64 doubles.
__device__ __forceinline__ void block_sum2(double& a, double& b, double* red) {
    a = warp_sum(a); b = warp_sum(b);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    if (l == 0) { red[w] = a; red[32 + w] = b; }
    __syncthreads();
    if (w == 0) {
        a = (l < nw) ? red[l] : 0.0;
        b = (l < nw) ? red[32 + l] : 0.0;
        a = warp_sum(a); b = warp_sum(b);
    }
}

// ------------------------------------------------------------------------------------------------ S1 per site
// Accumulate one link into the independent components of D = A - A^dag with sign sg (+1: U_mu(x-mu), -1: U_mu(x)).
//   d01 += sg (U01 - conj U10), d02 += sg (U02 - conj U20), d12 += sg (U12 - conj U21), im_j += sg Im U_jj
__device__ __forceinline__ void acc_link(const cplx (&u)[9], real sg, cplx& d01, cplx& d02, cplx& d12, real& i0, real& i1, real& i2) {
    d01.x = fma(sg, u[1].x - u[3].x, d01.x); d01.y = fma(sg, u[1].y + u[3].y, d01.y);
    d02.x = fma(sg, u[2].x - u[6].x, d02.x); d02.y = fma(sg, u[2].y + u[6].y, d02.y);
    d12.x = fma(sg, u[5].x - u[7].x, d12.x); d12.y = fma(sg, u[5].y + u[7].y, d12.y);
    i0 = fma(sg, u[0].y, i0); i1 = fma(sg, u[4].y, i1); i2 = fma(sg, u[8].y, i2);
}

// Delta(x) packed, plus this site's contributions to theta (Tr[Delta Delta^dag]) and F (sum_mu Re Tr U_mu(x)).
// ND = directions of the gauge condition (4 Landau, 3 Coulomb), a template parameter so that the loop over mu unrolls
// with all its loads free to be scheduled together (a run-time bound cost the fp32 pass A 17 %).
template <int NC, int ND>
__device__ __forceinline__ void delta_site_nd(const cplx* __restrict__ links, const Geom& G, long long x,
                                              cplx& f0, cplx& f1, cplx& f2, cplx& f3, double& th, double& fs) {
    cplx d01 = mk(0, 0), d02 = mk(0, 0), d12 = mk(0, 0);
    real i0 = 0, i1 = 0, i2 = 0, retr = 0;
#pragma unroll
    for (int mu = 0; mu < ND; mu++) {
        cplx u[9];
        load_link<NC>(links, G.V, mu, x, u);
        retr += u[0].x + u[4].x + u[8].x;
        acc_link(u, real(-1), d01, d02, d12, i0, i1, i2);
        load_link<NC>(links, G.V, mu, bwd(G, x, mu), u);
        acc_link(u, real(1), d01, d02, d12, i0, i1, i2);
    }
    // D_jj = 2i Im A_jj; Delta_jj = D_jj - Tr D / 3
    const real tr3 = real(2.0 / 3.0) * (i0 + i1 + i2);
    const real e0 = real(2) * i0 - tr3, e1 = real(2) * i1 - tr3, e2 = real(2) * i2 - tr3;
    f0 = d01; f1 = d02; f2 = d12; f3 = mk(e0, e1);
    th = (double)(real(2) * (cnorm2(d01) + cnorm2(d02) + cnorm2(d12)) + e0 * e0 + e1 * e1 + e2 * e2);
    fs = (double)retr;
}
template <int NC>
__device__ __forceinline__ void delta_site(const cplx* __restrict__ links, const Geom& G, long long x,
                                           cplx& f0, cplx& f1, cplx& f2, cplx& f3, double& th, double& fs) {
    if (G.nd == 4) delta_site_nd<NC, 4>(links, G, x, f0, f1, f2, f3, th, fs);
    else delta_site_nd<NC, 3>(links, G, x, f0, f1, f2, f3, th, fs);      // Coulomb gauge: the condition runs over mu = 0..2
}

template <int NC>
__global__ void __launch_bounds__(128) k_delta(const cplx* __restrict__ links, cplx* __restrict__ field, double2* __restrict__ partials,
                                               Geom G, const Ctl* __restrict__ ctl) {
    pdl_enter();
    if (ctl->done) return;
    __shared__ double red[64];
    const long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    cplx f0, f1, f2, f3;
    double th, fs;
    delta_site<NC>(links, G, x, f0, f1, f2, f3, th, fs);
    field[x] = f0; field[G.V + x] = f1; field[2 * G.V + x] = f2; field[3 * G.V + x] = f3;
    block_sum2(th, fs, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(th, fs);
}

// ------------------------------------------------------------------------------------------------ S5
// The S5 decision, by one thread: record (F, theta), raise the stop flag when theta < theta_tol (converged), max_iter
// updates have been applied, theta or F is not finite, or the stagnation guard fires.
__device__ __forceinline__ void s5_decide(Ctl* ctl, double2* hist, double theta, double F) {
    ctl->theta = theta; ctl->F = F;
    const int k = ctl->n_meas;
    if (k < ctl->hist_cap) hist[k] = make_double2(F, theta);
    ctl->n_meas = k + 1;
    if (!(isfinite(theta) && isfinite(F))) { ctl->nonfinite = 1; ctl->done = 1; }
    else if (theta < ctl->theta_tol) { ctl->converged = 1; ctl->done = 1; }
    else if (ctl->iters >= ctl->max_iter) { ctl->done = 1; }
    else if (ctl->stall_window > 0) {
        if (k == 0 || theta < 0.5 * ctl->theta_mark) { ctl->theta_mark = theta; ctl->stall_count = 0; }
        else if (++ctl->stall_count >= ctl->stall_window) { ctl->stalled = 1; ctl->done = 1; }
    }
}

// One block.  Sums the partials in a fixed order (strided per thread, then tree), writes F, theta, history,
// and raises the stop flag: theta < theta_tol (converged), or max_iter updates applied, or non-finite.
__global__ void __launch_bounds__(1024) k_finalize(const double2* __restrict__ partials, int n, Ctl* ctl, double2* hist, double inv3V, double inv12V) {
    pdl_enter();
    if (ctl->done) return;
    __shared__ double red[64];
    double a = 0, b = 0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) { double2 p = partials[i]; a += p.x; b += p.y; }
    block_sum2(a, b, red);
    if (threadIdx.x == 0) {
        s5_decide(ctl, hist, a * inv3V, b * inv12V);
    }
}

// ------------------------------------------------------------------------------------------------ S2 passes
struct FftTables {          // device pointers to per-axis tables (built on the host in long double)
    const cplx* tw[4];      // tw[mu][k] = exp(-2 pi i k / L_mu)
    const double* s[4];     // s[mu][p] = 4 sin^2(pi n/L_mu), n = frequency stored at position p after the forward DIF
    AxisPlan plan[4];       // stage radices of each axis (fft_tile.cuh)
};

enum { MODE_FWD = 0, MODE_INV = 1, MODE_DELTA_FWD = 2, MODE_INV_G = 3 };

// (x0,x1)-plane pass.  One CTA per (plane, group of NCOMP components); tile[c][x1][x0] with odd row stride.
//   MODE_FWD        field -> forward FFT over axes 0,1 -> field (in place)
//   MODE_DELTA_FWD  links -> Delta of the plane (S1, with theta/F partials) -> forward FFT -> field   [NCOMP = 4]
//   MODE_INV        field -> inverse FFT over axes 1,0 -> field (X, in place)
//   MODE_INV_G      field -> inverse FFT -> X -> g(x) rows 0,1 -> gbuf                               [NCOMP = 4]
template <int MODE, int NC>
__global__ void __launch_bounds__(256) k_fft01(cplx* __restrict__ field, const cplx* __restrict__ links, cplx* __restrict__ gbuf,
                                               double2* __restrict__ partials, Geom G, FftTables T, int ncomp, double half_alpha,
                                               const Ctl* __restrict__ ctl) {
    pdl_enter();
    if (ctl->done) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L0 = G.L[0], L1 = G.L[1];
    const int S1 = L0 + 1;                 // odd row stride: conflict-free for both axes
    const int S2 = S1 * L1;                // component stride
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw0 = tile + S2 * ncomp;
    cplx* tw1 = tw0 + L0;
    __shared__ double red[64];

    const int ngroups = 4 / ncomp;
    const long long plane = blockIdx.x / ngroups;           // = x2 + L2*x3
    const int c0 = (blockIdx.x % ngroups) * ncomp;
    const int lgP = G.lg[0] + G.lg[1];
    const int nP = 1 << lgP;
    const long long xbase = plane << lgP;

    for (int i = threadIdx.x; i < L0; i += blockDim.x) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += blockDim.x) tw1[i] = T.tw[1][i];

    if (MODE == MODE_DELTA_FWD) {
        double th = 0, fs = 0;
        for (int e = threadIdx.x; e < nP; e += blockDim.x) {
            cplx f0, f1, f2, f3;
            double t, f;
            delta_site<NC>(links, G, xbase + e, f0, f1, f2, f3, t, f);
            th += t; fs += f;
            const int o = (e & (L0 - 1)) + (e >> G.lg[0]) * S1;
            tile[o] = f0; tile[S2 + o] = f1; tile[2 * S2 + o] = f2; tile[3 * S2 + o] = f3;
        }
        block_sum2(th, fs, red);
        if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(th, fs);
    } else {
        const int ne = nP * ncomp;
        for (int e = threadIdx.x; e < ne; e += blockDim.x) {
            const int c = e >> lgP, r = e & (nP - 1);
            tile[c * S2 + (r & (L0 - 1)) + (r >> G.lg[0]) * S1] = field[(long long)(c0 + c) * G.V + xbase + r];
        }
    }
    __syncthreads();

    AxisXf a0, a1;
    a0.lgL = G.lg[0]; a0.strideK = 1;  a0.lgA = G.lg[1]; a0.strideA = S1; a0.nB = ncomp; a0.strideB = S2; a0.tw = tw0; a0.plan = T.plan[0];
    a1.lgL = G.lg[1]; a1.strideK = S1; a1.lgA = G.lg[0]; a1.strideA = 1;  a1.nB = ncomp; a1.strideB = S2; a1.tw = tw1; a1.plan = T.plan[1];
    if (MODE == MODE_FWD || MODE == MODE_DELTA_FWD) {
        fft_axis_forward(tile, a0);
        fft_axis_forward(tile, a1);
    } else {
        fft_axis_inverse(tile, a1);
        fft_axis_inverse(tile, a0);
    }

    if (MODE == MODE_INV_G) {
        for (int e = threadIdx.x; e < nP; e += blockDim.x) {
            const int o = (e & (L0 - 1)) + (e >> G.lg[0]) * S1;
            cplx g[9];
            build_g(tile[o], tile[S2 + o], tile[2 * S2 + o], tile[3 * S2 + o], (real)half_alpha, g);
#pragma unroll
            for (int c = 0; c < 6; c++) gbuf[(long long)c * G.V + xbase + e] = g[c];
        }
    } else {
        const int ne = nP * ncomp;
        for (int e = threadIdx.x; e < ne; e += blockDim.x) {
            const int c = e >> lgP, r = e & (nP - 1);
            field[(long long)(c0 + c) * G.V + xbase + r] = tile[c * S2 + (r & (L0 - 1)) + (r >> G.lg[0]) * S1];
        }
    }
}

// Axes 2,3 pass: forward, filter, inverse.  One CTA per (component, x1, chunk of C0 = 2^lgC consecutive x0);
// tile[x3][x2][i0].  scale = 16/V folds p2max and the 1/V of the inverse transform.          [north_star step 2]
__global__ void __launch_bounds__(256) k_fft23_mid(cplx* __restrict__ field, Geom G, FftTables T, int lgC, int S1, int S2, double scale,
                                                   const Ctl* __restrict__ ctl) {
    pdl_enter();
    if (ctl->done) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L2 = G.L[2], L3 = G.L[3];
    const int C0 = 1 << lgC;
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw2 = tile + S2 * L3;
    cplx* tw3 = tw2 + L2;
    double* s2 = reinterpret_cast<double*>(tw3 + L3);
    double* s3 = s2 + L2;

    const int lgChunks = G.lg[0] - lgC;
    const int chunk = blockIdx.x & ((1 << lgChunks) - 1);
    const int x1 = (blockIdx.x >> lgChunks) & (G.L[1] - 1);
    const int comp = blockIdx.x >> (lgChunks + G.lg[1]);
    const int p0base = chunk << lgC;
    cplx* gp = field + (long long)comp * G.V + p0base + ((long long)x1 << G.sh[1]);

    for (int i = threadIdx.x; i < L2; i += blockDim.x) { tw2[i] = T.tw[2][i]; s2[i] = T.s[2][i]; }
    for (int i = threadIdx.x; i < L3; i += blockDim.x) { tw3[i] = T.tw[3][i]; s3[i] = T.s[3][i]; }

    const int lg23 = G.lg[2] + G.lg[3];
    const int ne = C0 << lg23;
    for (int e = threadIdx.x; e < ne; e += blockDim.x) {
        const int i0 = e & (C0 - 1), r = e >> lgC;
        const int i2 = r & (L2 - 1), i3 = r >> G.lg[2];
        tile[i0 + i2 * S1 + i3 * S2] = gp[i0 + ((long long)i2 << G.sh[2]) + ((long long)i3 << G.sh[3])];
    }
    __syncthreads();

    AxisXf a2, a3;
    a2.lgL = G.lg[2]; a2.strideK = S1; a2.lgA = lgC; a2.strideA = 1; a2.nB = L3; a2.strideB = S2; a2.tw = tw2; a2.plan = T.plan[2];
    a3.lgL = G.lg[3]; a3.strideK = S2; a3.lgA = lgC; a3.strideA = 1; a3.nB = L2; a3.strideB = S1; a3.tw = tw3; a3.plan = T.plan[3];
    fft_axis_forward(tile, a2);
    fft_axis_forward(tile, a3);

    // S2b: X~ = (p2max / p2) Delta~ / V at the stored (digit-reversed) positions; zero mode -> 0
    const double s01_base = T.s[1][x1];
    for (int e = threadIdx.x; e < ne; e += blockDim.x) {
        const int i0 = e & (C0 - 1), r = e >> lgC;
        const int i2 = r & (L2 - 1), i3 = r >> G.lg[2];
        const double p2 = (T.s[0][p0base + i0] + s01_base) + (s2[i2] + s3[i3]);
        const double w = filter_weight(scale, p2);
        cplx* q = tile + i0 + i2 * S1 + i3 * S2;
        cplx v = *q;
        *q = cscale(v, (real)w);
    }
    __syncthreads();

    fft_axis_inverse(tile, a3);
    fft_axis_inverse(tile, a2);

    for (int e = threadIdx.x; e < ne; e += blockDim.x) {
        const int i0 = e & (C0 - 1), r = e >> lgC;
        const int i2 = r & (L2 - 1), i3 = r >> G.lg[2];
        gp[i0 + ((long long)i2 << G.sh[2]) + ((long long)i3 << G.sh[3])] = tile[i0 + i2 * S1 + i3 * S2];
    }
}

// ------------------------------------------------------------------------------------------------ S3 + S4
// S3+S4 with a stored g field (LGF_OPT_STORE_G): one thread per site reads rows 0,1 of g(x) and g(x+mu) from gbuf
// (96 B/site, written by pass C), rebuilds row 2 and rotates the four links of the site in place.  Each link (x,mu) is
// read and written by exactly one thread.
template <int NC>
__global__ void __launch_bounds__(128, 3) k_update_g(cplx* links, const cplx* __restrict__ gbuf, Geom G, Ctl* ctl) {
    pdl_enter();
    if (ctl->done) return;
    const long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long V = G.V;
    cplx g[9];
#pragma unroll
    for (int c = 0; c < 6; c++) g[c] = ldg2(gbuf + (long long)c * V + x);
    third_row(g);
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const long long xf = fwd(G, x, mu);
        cplx gp[9], u[9], r[9];
        load_link<NC, false>(links, V, mu, x, u);
#pragma unroll
        for (int c = 0; c < 6; c++) gp[c] = ldg2(gbuf + (long long)c * V + xf);
        third_row(gp);
        rotate_link<(NC == 6) ? 2 : 3>(g, u, gp, r);
        store_link<NC>(links, V, mu, x, r);
    }
    if (x == 0) ctl->iters = ctl->iters + 1;
}

// One thread per link, four warps per CTA = the four directions of 32 consecutive sites.  Thread (x, mu) builds
// g(x+mu) only; g(x) is what the mu = 0 thread of the site x-0 built (its forward neighbour is x), handed over
// through shared memory: 4 Gram-Schmidt per site instead of 5 (one thread per site) or 8 (no sharing).
// A CTA covers whole x0 rows (NS = max(32, L0) sites, 4 NS threads), so the site x-0 is always in the same CTA.
// Measured on B200 at 32^4 (CUDA events per launch): 149 us at 5 CTAs/SM (96 registers), 157 at 4, 157 at 6 (spills),
// against 161 for one thread per site (k_update<NC,0>, 12 warps/SM); the IEEE 1/sqrt costs nothing measurable.
// > 0: each thread prefetches into L2 the link its counterpart that many CTAs ahead will load.  Measured on B200 at 32^4
// with 740 (= one resident wave of 5 CTAs x 148 SMs): fp32 83.7 against 87.7 us, fp64 148.3 against 145 us (1480: 153,
// 2960: 169) -- on in the fp32 build only.
#ifndef LGF_UPDQ_PREFETCH
#ifdef LGF_F32
#define LGF_UPDQ_PREFETCH 740
#else
#define LGF_UPDQ_PREFETCH 0
#endif
#endif
#ifndef LGF_UPDQ_MINB64
#define LGF_UPDQ_MINB64 3
#endif
#ifndef LGF_UPDQ_MINB
#define LGF_UPDQ_MINB 5
#endif
// ACC: the mu = 1 thread of each site also accumulates the total gauge transformation, Gacc(x) <- g(x) Gacc(x)
// (rows 0,1 in gacc, 6 V-arrays; mixed precision, lgf_api.cu): +2 x 6 complex per site.
template <int NC, int NS, int ACC = 0, int LGB = 0>      // NS = sites per CTA = max(32, L0): 4 * NS threads, thread = (mu, site)
__global__ void __launch_bounds__(4 * NS, (NS == 32) ? LGF_UPDQ_MINB : ((NS == 64) ? LGF_UPDQ_MINB64 : 1)) k_update_quad(cplx* links, const cplx* __restrict__ src, Geom G,
                                                                                       double half_alpha, Ctl* ctl, cplx* __restrict__ gacc = nullptr) {
    pdl_enter();
    if (ctl->done) return;
    __shared__ cplx sg[9][NS];
    const int st = threadIdx.x % NS, mu = threadIdx.x / NS;
    const long long V = G.V;
    // LGB > 0 (large lattices, NS = L0: a CTA is one x0 row): the rows are walked x1 fastest, then x2 inside a band of
    // 2^LGB values, then x3, then the bands -- so that X(x+3), first fetched as the forward neighbour of x, is still in L2
    // when the row x+3 itself is updated 2^LGB * L0 * L1 sites later.  In plain lexicographic order that takes L0 L1 L2
    // sites, 218 MB of link traffic at 64^4, and ncu showed the whole X field read from DRAM twice (8.59 GB of reads
    // against 7.52 GB algorithmic).  32-bit shifts and masks only: the row index heads every CTA's dependency chain.
    unsigned row = blockIdx.x;
    if constexpr (LGB > 0) {
        const unsigned x1 = row & (G.L[1] - 1);
        unsigned t = row >> G.lg[1];
        const unsigned x2l = t & ((1u << LGB) - 1); t >>= LGB;
        const unsigned x3 = t & (G.L[3] - 1);
        const unsigned bnd = t >> G.lg[3];
        row = x1 + (((bnd << LGB) + x2l) << G.lg[1]) + (x3 << (G.lg[1] + G.lg[2]));
    }
    const long long x = (long long)row * NS + st;
    const long long xf = fwd(G, x, mu);
    cplx g[9], gp[9], u[9], r[9];
#if LGF_UPDQ_PREFETCH
    {   // the link this thread's counterpart LGF_UPDQ_PREFETCH CTAs ahead will load: DRAM -> L2 now
        const long long xp = x + (long long)LGF_UPDQ_PREFETCH * NS;
        if (xp < V && prefetch_lane()) {
            const cplx* q = links + (long long)(mu * NC) * V + xp;
#pragma unroll
            for (int c = 0; c < NC; c++) prefetch_line_l2(q + (long long)c * V);
        }
    }
#endif
    load_link<NC, false>(links, V, mu, x, u);
    build_g(ldc_field(src + xf), ldc_field(src + V + xf), ldc_field(src + 2 * V + xf), ldc_field(src + 3 * V + xf), (real)half_alpha, gp);
    if (mu == 0) {
        const int m = G.L[0] - 1;                             // L0 <= NS: the x0 row of a site lies inside its CTA
        const int dst = (st & ~m) | ((st + 1) & m);           // the slot of site x+0 (same row, periodic)
#pragma unroll
        for (int c = 0; c < 9; c++) sg[c][dst] = gp[c];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 9; c++) g[c] = sg[c][st];
    rotate_link<(NC == 6) ? 2 : 3>(g, u, gp, r);
    store_link<NC>(links, V, mu, x, r);
    if (ACC && mu == 1) {
        cplx a[9];
#pragma unroll
        for (int c = 0; c < 6; c++) a[c] = gacc[(long long)c * V + x];
        third_row(a);
#pragma unroll
        for (int i = 0; i < 2; i++)
#pragma unroll
            for (int j = 0; j < 3; j++) {
                cplx t = cmul(g[3 * i], a[j]);
                t = cfma(g[3 * i + 1], a[3 + j], t);
                t = cfma(g[3 * i + 2], a[6 + j], t);
                gacc[(long long)(3 * i + j) * V + x] = t;
            }
    }
    if (x == 0 && mu == 0) ctl->iters = ctl->iters + 1;
}

// Gacc(x) = 1 (rows 0,1)
__global__ void __launch_bounds__(256) k_init_gacc(cplx* __restrict__ gacc, long long V) {
    const long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= V) return;
#pragma unroll
    for (int c = 0; c < 6; c++) gacc[(long long)c * V + x] = mk((c == 0 || c == 4) ? real(1) : real(0), real(0));
}

#ifndef LGF_F32
// ---- mixed precision (fp64 build only): the fp32 shadow context works on a float copy of the links and accumulates
// the gauge transformation; the fp64 links then receive it in one step, U_mu(x) <- G(x) U_mu(x) G(x+mu)^dagger, with G
// re-orthonormalised in double, so the result is an exact (to fp64 rounding) gauge copy of the fp64 input.
__global__ void __launch_bounds__(256) k_demote(const double2* __restrict__ src, float2* __restrict__ dst, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { const double2 v = __ldg(src + i); dst[i] = make_float2((float)v.x, (float)v.y); }
}
__device__ __forceinline__ void load_gacc64(const float2* __restrict__ gacc, long long V, long long x, cplx (&g)[9]) {
    cplx m[6];
#pragma unroll
    for (int c = 0; c < 6; c++) { const float2 v = __ldg(gacc + (long long)c * V + x); m[c] = mk((double)v.x, (double)v.y); }
    // row Gram-Schmidt in double (the same projection as S3), third row = conj(u x v)
    const double r0 = 1.0 / sqrt(cnorm2(m[0]) + cnorm2(m[1]) + cnorm2(m[2]));
    g[0] = cscale(m[0], r0); g[1] = cscale(m[1], r0); g[2] = cscale(m[2], r0);
    cplx ip = ccmul(g[0], m[3]);
    ip = cadd(ip, ccmul(g[1], m[4]));
    ip = cadd(ip, ccmul(g[2], m[5]));
    const cplx v0 = cfnma(ip, g[0], m[3]), v1 = cfnma(ip, g[1], m[4]), v2 = cfnma(ip, g[2], m[5]);
    const double r1 = 1.0 / sqrt(cnorm2(v0) + cnorm2(v1) + cnorm2(v2));
    g[3] = cscale(v0, r1); g[4] = cscale(v1, r1); g[5] = cscale(v2, r1);
    third_row(g);
}
template <int NC>
__global__ void __launch_bounds__(128) k_apply_gacc(cplx* links, const float2* __restrict__ gacc, Geom G) {
    const int mu = blockIdx.x & 3;
    const long long x = (long long)(blockIdx.x >> 2) * 128 + threadIdx.x;
    cplx g[9], gp[9], u[9], r[9];
    load_link<NC, false>(links, G.V, mu, x, u);
    load_gacc64(gacc, G.V, x, g);
    load_gacc64(gacc, G.V, fwd(G, x, mu), gp);
    rotate_link<(NC == 6) ? 2 : 3>(g, u, gp, r);
    store_link<NC>(links, G.V, mu, x, r);
}
#endif

// ------------------------------------------------------------------------------------------------ boundary helpers
// canonical [x][mu][3][3] complex (array of structs; ne = 9 entries per link, or ne = 6: the two-row host format
// [x][mu][2][3]) -> structure of arrays; one thread per (x, mu).  ne >= NC.
template <int NC>
__global__ void __launch_bounds__(256) k_layout_in(const dcplx* __restrict__ aos, cplx* __restrict__ links, long long V, long long x_off, long long n_sites, int ne) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_sites * 4) return;
    const int mu = (int)(i / n_sites);
    const long long xl = i % n_sites;
    const dcplx* s = aos + (xl * 4 + mu) * ne;
    cplx* d = links + (long long)(mu * NC) * V + x_off + xl;
#pragma unroll
    for (int c = 0; c < NC; c++) d[(long long)c * V] = mk((real)s[c].x, (real)s[c].y);
}
template <int NC>
__global__ void __launch_bounds__(256) k_layout_out(const cplx* __restrict__ links, dcplx* __restrict__ aos, long long V, long long x_off, long long n_sites, int ne) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_sites * 4) return;
    const int mu = (int)(i / n_sites);
    const long long xl = i % n_sites;
    cplx u[9];
    load_link<NC>(links, V, mu, x_off + xl, u);
    dcplx* d = aos + (xl * 4 + mu) * ne;
#pragma unroll
    for (int c = 0; c < 9; c++) if (c < ne) d[c] = make_double2((double)u[c].x, (double)u[c].y);
}

// packed 4-component field -> full 3x3 anti-Hermitian matrices [x][3][3]
__device__ __forceinline__ dcplx widen(cplx v) { return make_double2((double)v.x, (double)v.y); }
__global__ void __launch_bounds__(256) k_unpack_field(const cplx* __restrict__ field, dcplx* __restrict__ out, long long V, long long x_off, long long n_sites) {
    const long long xl = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (xl >= n_sites) return;
    const long long x = x_off + xl;
    const dcplx f0 = widen(field[x]), f1 = widen(field[V + x]), f2 = widen(field[2 * V + x]), f3 = widen(field[3 * V + x]);
    dcplx* d = out + xl * 9;
    d[0] = make_double2(0, f3.x); d[1] = f0; d[2] = f1;
    d[3] = make_double2(-f0.x, f0.y); d[4] = make_double2(0, f3.y); d[5] = f2;
    d[6] = make_double2(-f1.x, f1.y); d[7] = make_double2(-f2.x, f2.y); d[8] = make_double2(0, -(f3.x + f3.y));
}
// g rows 0,1 (6 arrays) -> full [x][3][3];  or rebuilt from the packed X field when from_x != 0
__global__ void __launch_bounds__(256) k_unpack_g(const cplx* __restrict__ src, int from_x, double half_alpha, dcplx* __restrict__ out, long long V,
                                                  long long x_off, long long n_sites) {
    const long long xl = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (xl >= n_sites) return;
    const long long x = x_off + xl;
    cplx g[9];
    if (from_x) build_g(src[x], src[V + x], src[2 * V + x], src[3 * V + x], (real)half_alpha, g);
    else {
#pragma unroll
        for (int c = 0; c < 6; c++) g[c] = src[(long long)c * V + x];
        third_row(g);
    }
    dcplx* d = out + xl * 9;
#pragma unroll
    for (int c = 0; c < 9; c++) d[c] = widen(g[c]);
}

// 3x3 product helpers for the plaquette (not on the hot path)
__device__ __forceinline__ void mm(const cplx (&a)[9], const cplx (&b)[9], cplx (&r)[9]) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cplx s = cmul(a[3 * i], b[j]);
            s = cfma(a[3 * i + 1], b[3 + j], s);
            s = cfma(a[3 * i + 2], b[6 + j], s);
            r[3 * i + j] = s;
        }
}
__device__ __forceinline__ void mmd(const cplx (&a)[9], const cplx (&b)[9], cplx (&r)[9]) {  // a * b^dag
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cplx s = cmulc(a[3 * i], b[3 * j]);
            s = cfmac(a[3 * i + 1], b[3 * j + 1], s);
            s = cfmac(a[3 * i + 2], b[3 * j + 2], s);
            r[3 * i + j] = s;
        }
}
// sum over the 6 planes of Re Tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag]; partials[block].x
template <int NC>
__global__ void __launch_bounds__(128) k_plaquette(const cplx* __restrict__ links, double2* __restrict__ partials, Geom G) {
    __shared__ double red[64];
    const long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double p = 0, z = 0;
    for (int mu = 0; mu < 4; mu++)
        for (int nu = mu + 1; nu < 4; nu++) {
            cplx a[9], b[9], c[9], d[9];
            load_link<NC>(links, G.V, mu, x, a);
            load_link<NC>(links, G.V, nu, fwd(G, x, mu), b);
            mm(a, b, c);
            load_link<NC>(links, G.V, mu, fwd(G, x, nu), a);
            mmd(c, a, d);
            load_link<NC>(links, G.V, nu, x, b);
            mmd(d, b, c);
            p += (double)(c[0].x + c[4].x + c[8].x);
        }
    block_sum2(p, z, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(p, 0.0);
}
__global__ void __launch_bounds__(256) k_sum_partials(const double2* __restrict__ partials, int n, double* out) {
    __shared__ double red[64];
    double a = 0, b = 0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) { double2 p = partials[i]; a += p.x; b += p.y; }
    block_sum2(a, b, red);
    if (threadIdx.x == 0) { out[0] = a; out[1] = b; }
}

#ifndef LGF_F32
// streaming double2 copy: the measured-peak yardstick (grid-stride, 4 independent 16 B loads per thread per trip)
__global__ void __launch_bounds__(256) k_copy(double2* __restrict__ dst, const double2* __restrict__ src, long long n) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n; i += 4 * stride) {
        double2 a = __ldg(src + i), b = __ldg(src + i + stride), c = __ldg(src + i + 2 * stride), d = __ldg(src + i + 3 * stride);
        dst[i] = a; dst[i + stride] = b; dst[i + 2 * stride] = c; dst[i + 3 * stride] = d;
    }
    for (; i < n; i += stride) dst[i] = __ldg(src + i);
}

// 24 SoA streams, one double2 per thread and stream: the link kernels' access pattern without their arithmetic
template <int RW>
__global__ void __launch_bounds__(128) k_streams(double2* __restrict__ a, long long V, double2* __restrict__ sink) {
    const long long x = (long long)blockIdx.x * 128 + threadIdx.x;
    double2 v[24];
#pragma unroll
    for (int c = 0; c < 24; c++) v[c] = __ldg(a + (long long)c * V + x);
    if (RW) {
#pragma unroll
        for (int c = 0; c < 24; c++) a[(long long)c * V + x] = make_double2(v[c].y, v[c].x);
    } else {
        double s = 0;
#pragma unroll
        for (int c = 0; c < 24; c++) s += v[c].x * v[c].y;
        if (s == 1.2345e300) sink[0] = make_double2(s, s);      // never true for finite data: keeps the loads alive
    }
}

// FP64 FMA yardstick: every thread runs 8 independent chains of dependent DFMAs in registers (no memory traffic);
// 2 * 8 * iters flops per thread.  The second roof of the FFT passes.
__global__ void __launch_bounds__(256) k_fma64(double* __restrict__ sink, int iters, double a, double b) {
    double x0 = threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
#pragma unroll 4
    for (int i = 0; i < iters; i++) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 1.2345e300) sink[0] = s;                                 // never true: keeps the chains alive
}

#endif  // LGF_F32

}  // namespace lgf
