// slab.cuh -- kernels of the slab-decomposed iteration (the paper's CPU comparator is this
// decomposition over MPI + PFFT).
//
// The lattice is cut along axis 3 into P slabs of L3/P time slices; rank r owns the sites with x3 in [r L3/P, (r+1) L3/P)
// in its own workspace: links [4][NC][Vloc], field [4][Vloc], x = x0 + L0 (x1 + L1 (x2 + L2 x3loc)).  One iteration:
//   halo 1    U_3 of the last slice of rank r-1  ->  halo_u of rank r                       (NC * S complex, S = L0 L1 L2)
//   S1        k_delta_slab: Delta, theta/F partials (the backward neighbour along axis 3 of slice 0 comes from halo_u)
//   pass A    forward FFT over axes 0,1, local (the plane passes of kernels.cuh on the local lattice)
//   transpose k_slab_scatter: rank r writes the part of its field with x1 in rank s's range straight into rank s's
//             transposed buffer fieldT [4][L3][L2][L1/P][L0] -- a store to peer memory over NVLink when the ranks are GPUs
//   pass B    axes 2,3 forward, p2max/p2 filter, inverse, local on the transposed lattice (L0, L1/P, L2, L3)
//   transpose k_slab_gather: the mirror image, fieldT of rank r -> field of every rank s
//   pass C    inverse FFT over axes 1,0, local
//   halo 2    X of the first slice of rank r+1  ->  halo_x of rank r                          (4 * S complex)
//   S3+S4     k_update_slab: as k_update_quad; X(x+3) of the last slice comes from halo_x
// Everything else (arithmetic, stored FFT order, reductions, stop flag) is that of the single-context path.
#pragma once
#include "kernels.cuh"

namespace lgf {

constexpr int SLAB_MAX_RANKS = 16;
struct SlabPeers { cplx* p[SLAB_MAX_RANKS]; };      // one buffer per rank (peer pointers when the ranks are GPUs)

// S1 on a slab: delta_site_nd<NC,4> with the axis-3 backward neighbour of slice 0 read from halo_u (NC arrays of S).
template <int NC>
__global__ void __launch_bounds__(128) k_delta_slab(const cplx* __restrict__ links, const cplx* __restrict__ halo_u, cplx* __restrict__ field,
                                                    double2* __restrict__ partials, Geom G, const Ctl* __restrict__ ctl) {
    if (ctl->done) return;
    __shared__ double red[64];
    const long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long S = 1LL << G.sh[3];
    cplx d01 = mk(0, 0), d02 = mk(0, 0), d12 = mk(0, 0);
    real i0 = 0, i1 = 0, i2 = 0, retr = 0;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        cplx u[9];
        load_link<NC>(links, G.V, mu, x, u);
        retr += u[0].x + u[4].x + u[8].x;
        acc_link(u, real(-1), d01, d02, d12, i0, i1, i2);
        if (mu == 3 && x < S) {                          // slice 0 of the slab: U_3(x-3) lives on the rank below
#pragma unroll
            for (int c = 0; c < NC; c++) u[c] = __ldg(halo_u + (long long)c * S + x);
            if (NC == 6) third_row(u);
        } else load_link<NC>(links, G.V, mu, bwd(G, x, mu), u);
        acc_link(u, real(1), d01, d02, d12, i0, i1, i2);
    }
    const real tr3 = real(2.0 / 3.0) * (i0 + i1 + i2);
    const real e0 = real(2) * i0 - tr3, e1 = real(2) * i1 - tr3, e2 = real(2) * i2 - tr3;
    field[x] = d01; field[G.V + x] = d02; field[2 * G.V + x] = d12; field[3 * G.V + x] = mk(e0, e1);
    double th = (double)(real(2) * (cnorm2(d01) + cnorm2(d02) + cnorm2(d12)) + e0 * e0 + e1 * e1 + e2 * e2);
    double fs = (double)retr;
    block_sum2(th, fs, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(th, fs);
}

// Transposes.  Local lattice of rank r: (L0, L1, L2, L3l), transposed lattice of rank s: (L0, L1l, L2, L3); L1l = L1/P,
// L3l = L3/P.  One thread per (x0, x1, x2, x3l) of the SOURCE rank; four components.
//   scatter: field_r[c][x0, x1, x2, x3l]  ->  fieldT_s[c][x0, x1 mod L1l, x2, x3l + r L3l],  s = x1 / L1l
__global__ void __launch_bounds__(256) k_slab_scatter(const cplx* __restrict__ field, SlabPeers dstT, int rank, int lg0, int lg1, int lg2, int lg3l,
                                                      int lgP, const Ctl* __restrict__ ctl) {
    if (ctl->done) return;
    const long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long Vl = 1LL << (lg0 + lg1 + lg2 + lg3l);
    if (x >= Vl) return;
    const int lg1l = lg1 - lgP;
    const int x0 = (int)(x & ((1 << lg0) - 1)), x1 = (int)(x >> lg0) & ((1 << lg1) - 1), x2 = (int)(x >> (lg0 + lg1)) & ((1 << lg2) - 1);
    const int x3l = (int)(x >> (lg0 + lg1 + lg2));
    const int s = x1 >> lg1l;
    const long long y = x0 + ((long long)(x1 & ((1 << lg1l) - 1)) << lg0) + ((long long)x2 << (lg0 + lg1l)) +
                        ((long long)(x3l + (rank << lg3l)) << (lg0 + lg1l + lg2));
    cplx* d = dstT.p[s];
#pragma unroll
    for (int c = 0; c < 4; c++) d[(long long)c * Vl + y] = field[(long long)c * Vl + x];      // the transposed lattice has Vl sites too
}
//   gather: fieldT_r[c][x0, x1l, x2, x3]  ->  field_s[c][x0, x1l + r L1l, x2, x3 mod L3l],  s = x3 / L3l
__global__ void __launch_bounds__(256) k_slab_gather(const cplx* __restrict__ fieldT, SlabPeers dst, int rank, int lg0, int lg1, int lg2, int lg3l,
                                                     int lgP, const Ctl* __restrict__ ctl) {
    if (ctl->done) return;
    const long long y = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long Vl = 1LL << (lg0 + lg1 + lg2 + lg3l);
    if (y >= Vl) return;
    const int lg1l = lg1 - lgP;
    const int x0 = (int)(y & ((1 << lg0) - 1)), x1l = (int)(y >> lg0) & ((1 << lg1l) - 1), x2 = (int)(y >> (lg0 + lg1l)) & ((1 << lg2) - 1);
    const int x3 = (int)(y >> (lg0 + lg1l + lg2));
    const int s = x3 >> lg3l;
    const long long x = x0 + ((long long)(x1l + (rank << lg1l)) << lg0) + ((long long)x2 << (lg0 + lg1)) +
                        ((long long)(x3 & ((1 << lg3l) - 1)) << (lg0 + lg1 + lg2));
    cplx* d = dst.p[s];
#pragma unroll
    for (int c = 0; c < 4; c++) d[(long long)c * Vl + x] = fieldT[(long long)c * Vl + y];
}

// S3+S4 on a slab: k_update_quad with X(x+3) of the last local slice read from halo_x (4 arrays of S).
template <int NC, int NS>
__global__ void __launch_bounds__(4 * NS, (NS == 32) ? 4 : 2) k_update_slab(cplx* links, const cplx* __restrict__ src, const cplx* __restrict__ halo_x, Geom G,
                                                                             double half_alpha, Ctl* ctl, int count_iters) {
    if (ctl->done) return;
    __shared__ cplx sg[9][NS];
    const int st = threadIdx.x % NS, mu = threadIdx.x / NS;
    const long long V = G.V, S = 1LL << G.sh[3];
    const long long x = (long long)blockIdx.x * NS + st;
    cplx g[9], gp[9], u[9], r[9];
    load_link<NC, false>(links, V, mu, x, u);
    if (mu == 3 && x >= V - S) {                         // last slice of the slab: X(x+3) lives on the rank above
        const long long xs = x - (V - S);
        build_g(__ldg(halo_x + xs), __ldg(halo_x + S + xs), __ldg(halo_x + 2 * S + xs), __ldg(halo_x + 3 * S + xs), (real)half_alpha, gp);
    } else {
        const long long xf = fwd(G, x, mu);
        build_g(ldc_field(src + xf), ldc_field(src + V + xf), ldc_field(src + 2 * V + xf), ldc_field(src + 3 * V + xf), (real)half_alpha, gp);
    }
    if (mu == 0) {
        const int m = G.L[0] - 1;
        const int dst = (st & ~m) | ((st + 1) & m);
#pragma unroll
        for (int c = 0; c < 9; c++) sg[c][dst] = gp[c];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 9; c++) g[c] = sg[c][st];
    rotate_link<(NC == 6) ? 2 : 3>(g, u, gp, r);
    store_link<NC>(links, V, mu, x, r);
    if (count_iters && x == 0 && mu == 0) ctl->iters = ctl->iters + 1;
}

}  // namespace lgf
