// fft_fast.cuh -- compile-time-sized FFT passes for the common lattice extents (L = 16, 32, 64 per axis).
//
// Same arithmetic and the same stored (digit-reversed) order as the generic passes of kernels.cuh/fft_tile.cuh --
// the per-axis stage radices are those of AxisPlan (lgf_api.cu make_plan) -- but organised to cross shared memory
// as few times as possible (ncu, profiles/r01_README.md: the generic passes are shared-memory/latency-bound):
//   * every extent is two stages (R1, R2); the first stage of a pass takes its inputs straight from global
//     memory (or from the Delta tile) and the last stage writes straight to global memory;
//   * when R2(a) * R1(b) <= 16 the last stage of axis a and the first stage of axis b are done on one 16-point
//     register block (one shared-memory round trip instead of two);
//   * in the middle pass the last forward stage of axis 3, the p2max/p2 filter and the first inverse stage of
//     axis 3 act on the same registers.
// Shared-memory round trips per point at 32^4:  pass A 3 (was 5), pass B 4 (was 10), pass C 2 (was 5).
// Everything (extents, strides, work counts) is a template parameter, so all loops unroll and index arithmetic
// folds into immediates.
#pragma once
#include <type_traits>
#include <cooperative_groups.h>
#include "kernels.cuh"

// resident CTAs per SM the passes are compiled for (register cap = 65536 / (NT * MINB)).  Measured on B200 at 32^4
// (CUDA events per launch): pass A 118.9 us at 1 CTA/SM, 107.7 at 2, 143.2 at 3 (spills); pass B 66.0 / 47.3 / 59.3.
#ifndef LGF_FA_MINB_DELTA
#define LGF_FA_MINB_DELTA 2
#endif
// 1: pass A prefetches the own links of a thread's next site into L2 (prefetch.global.L2) before it works on the current
// one.  Measured on B200 at 32^4: fp32 61.5 against 65.8 us, fp64 115.5 against 106 us (the extra L1TEX requests cost
// more than the latency they save) -- so it is on in the fp32 build only.
#ifndef LGF_FA_PREFETCH_NEXT
#ifdef LGF_F32
#define LGF_FA_PREFETCH_NEXT 1
#else
#define LGF_FA_PREFETCH_NEXT 0
#endif
#endif
#ifndef LGF_FA_MINB_MID
#define LGF_FA_MINB_MID 2
#endif
#ifndef LGF_FA_MINB_INV
#define LGF_FA_MINB_INV 1
#endif

namespace lgf {

// A group of NT threads that works on one tile: thread index within the group and the named barrier the group
// synchronises on.  A whole CTA is the group {threadIdx.x, 0} (bar.sync 0 over all threads = __syncthreads()).
struct Grp { int tid; int bar; };
template <int NT> __device__ __forceinline__ void gsync(const Grp& g) {
    asm volatile("bar.sync %0, %1;" ::"r"(g.bar), "n"(NT) : "memory");
}
// Compile-time group: BAR = 0 is the whole CTA (__syncthreads), else a named barrier over NT threads.
template <int NT, int BAR> __device__ __forceinline__ void gsync_c() {
    if constexpr (BAR == 0) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"n"(BAR), "n"(NT) : "memory");
}

// Two-stage plan of an axis of length 2^LG (LG = 4, 5, 6); B = axis 1 or 3.  Must agree with make_plan().
template <int LG, bool B> struct Plan2 {
    static_assert(LG >= 4 && LG <= 6, "fast FFT passes cover L = 16, 32, 64");
    static constexpr int LG1 = (LG == 4) ? 2 : ((LG == 5) ? (B ? 2 : 3) : 3);
    static constexpr int LG2 = LG - LG1;
    static constexpr int R1 = 1 << LG1, R2 = 1 << LG2, L = 1 << LG;
};

// Plan of an axis inside pass B (axes 2,3): as Plan2, except that a 64-point axis is 16 x 4 (axis 2) or 4 x 16 (axis 3)
// with the radix-16 stage done as 4 x 4 in registers (bfly16: the stored order of the generic plan [4,4,4], lgf_api.cu
// make_plan), so that the last stage of axis 2 and the first of axis 3 are always one 16-point register block: the tile
// crosses shared memory 4 times per direction... 8 passes in all at 64 x 64 instead of 12 with 8 x 8.
template <int LG, bool B> struct PlanM {
    static_assert(LG >= 4 && LG <= 6, "fast FFT passes cover L = 16, 32, 64");
    static constexpr int LG1 = (LG == 6) ? (B ? 2 : 4) : Plan2<LG, B>::LG1;
    static constexpr int LG2 = LG - LG1;
    static constexpr int R1 = 1 << LG1, R2 = 1 << LG2, L = 1 << LG;
};

// Forward stage on registers: y = DFT_R(v), then y_k *= tw[k*t]  (t = j * L/N: W_N^{jk} = tw[k t]).
// Inverse stage: v_k *= conj(tw[k t]), then y = IDFT_R(v).  Slot s of a radix-16 butterfly holds frequency slot_freq(s).
template <int R, bool INV, bool TW>
__device__ __forceinline__ void stage_regs(cplx (&v)[R], const cplx* __restrict__ tw, int t) {
    if constexpr (INV) {
        if constexpr (TW) {
#pragma unroll
            for (int k = 1; k < R; k++) v[k] = cmulc(v[k], tw[slot_freq<R>(k) * t]);
        }
        bfly<R, true>(v);
    } else {
        bfly<R, false>(v);
        if constexpr (TW) {
#pragma unroll
            for (int k = 1; k < R; k++) v[k] = cmul(v[k], tw[slot_freq<R>(k) * t]);
        }
    }
}

// One 1-D stage on a shared tile: element m of work item at p[m * stride].
template <int R, bool INV, bool TW>
__device__ __forceinline__ void stage_smem(cplx* __restrict__ p, int stride, const cplx* __restrict__ tw, int t) {
    cplx v[R];
#pragma unroll
    for (int m = 0; m < R; m++) v[m] = p[m * stride];
    stage_regs<R, INV, TW>(v, tw, t);
#pragma unroll
    for (int m = 0; m < R; m++) p[m * stride] = v[m];
}

// Fused block: the last stage of axis a (radix RA, contiguous sub-blocks, no twiddles) and the first stage of axis b
// (radix RB, sub-length = full extent, twiddles tw[kb * jb]) on an RB x RA register block.
// Element (ma, mb) at p[ma * sa + mb * sb].  Forward: a then b.  Inverse: b then a.
template <int RA, int RB, bool INV>
__device__ __forceinline__ void block_smem(cplx* __restrict__ p, int sa, int sb, const cplx* __restrict__ twb, int jb) {
    cplx v[RB][RA];
#pragma unroll
    for (int mb = 0; mb < RB; mb++)
#pragma unroll
        for (int ma = 0; ma < RA; ma++) v[mb][ma] = p[ma * sa + mb * sb];
    if constexpr (!INV) {
#pragma unroll
        for (int mb = 0; mb < RB; mb++) bfly<RA, false>(v[mb]);
    }
#pragma unroll
    for (int ma = 0; ma < RA; ma++) {
        cplx c[RB];
#pragma unroll
        for (int mb = 0; mb < RB; mb++) c[mb] = v[mb][ma];
        stage_regs<RB, INV, true>(c, twb, jb);
#pragma unroll
        for (int mb = 0; mb < RB; mb++) v[mb][ma] = c[mb];
    }
    if constexpr (INV) {
#pragma unroll
        for (int mb = 0; mb < RB; mb++) bfly<RA, true>(v[mb]);
    }
#pragma unroll
    for (int mb = 0; mb < RB; mb++)
#pragma unroll
        for (int ma = 0; ma < RA; ma++) p[ma * sa + mb * sb] = v[mb][ma];
}

// ---------------------------------------------------------------------------------------------------------------
// The middle stages of a 2-D transform of NCOMP tiles t[c][b][a] (row stride S odd, component stride SC), i.e.
// everything between the first stage of axis a and the last stage of axis b (forward), or the mirror (inverse).
// Ends with a group barrier.
template <int LGA, int LGB, int NCOMP, int NT, bool INV>
__device__ __forceinline__ void plane_middle(cplx* __restrict__ t, const cplx* __restrict__ twb, const Grp& g) {
    using PA = Plan2<LGA, false>;
    using PB = Plan2<LGB, true>;
    constexpr int LA = PA::L, LB = PB::L, S = LA + 1, SC = S * LB;
    if constexpr (PA::R2 * PB::R1 <= 16) {
        // lanes run over jb (rows, odd stride S: conflict-free), then over the a-blocks
        constexpr int NW = NCOMP * PA::R1 * PB::R2;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + g.tid;
            if (NW % NT == 0 || w < NW) {
                const int jb = w % PB::R2, ba = (w / PB::R2) % PA::R1, c = w / (PB::R2 * PA::R1);
                block_smem<PA::R2, PB::R1, INV>(t + c * SC + jb * S + ba * PA::R2, 1, PB::R2 * S, twb, jb);
            }
        }
        gsync<NT>(g);
    } else {
        // a stage 2 (contiguous sub-blocks of R2 points, no twiddles): lanes over rows
        auto a2 = [&]() {
            constexpr int NW = NCOMP * PA::R1 * LB;
#pragma unroll
            for (int w0 = 0; w0 < NW; w0 += NT) {
                const int w = w0 + g.tid;
                if (NW % NT == 0 || w < NW) {
                    const int xb = w % LB, ba = (w / LB) % PA::R1, c = w / (LB * PA::R1);
                    stage_smem<PA::R2, INV, false>(t + c * SC + xb * S + ba * PA::R2, 1, nullptr, 0);
                }
            }
            gsync<NT>(g);
        };
        // b stage 1 (sub-length LB, twiddles tw[k jb]): lanes over columns
        auto b1 = [&]() {
            constexpr int NW = NCOMP * LA * PB::R2;
#pragma unroll
            for (int w0 = 0; w0 < NW; w0 += NT) {
                const int w = w0 + g.tid;
                if (NW % NT == 0 || w < NW) {
                    const int xa = w % LA, jb = (w / LA) % PB::R2, c = w / (LA * PB::R2);
                    stage_smem<PB::R1, INV, true>(t + c * SC + jb * S + xa, PB::R2 * S, twb, jb);
                }
            }
            gsync<NT>(g);
        };
        if constexpr (INV) { b1(); a2(); } else { a2(); b1(); }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Forward FFT over axes 0,1 of the 4 component tiles t[c][x1][x0] (row stride L0+1), last stage written straight
// to field (component c at field + c*V, plane base xbase).  The tile must be complete (caller syncs before).
template <int LG0, int LG1, int NT, int NCOMP = 4>
__device__ __forceinline__ void plane_forward_store(cplx* __restrict__ tile, const cplx* __restrict__ tw0, const cplx* __restrict__ tw1,
                                                    cplx* __restrict__ field, long long V, long long xbase, const Grp& g) {
    using PA = Plan2<LG0, false>;
    using PB = Plan2<LG1, true>;
    constexpr int L0 = PA::L, L1 = PB::L, S = L0 + 1, SC = S * L1;
    // a stage 1: points a = ja + m R2, twiddles tw0[k ja]; lanes over rows
    {
        constexpr int NW = NCOMP * PA::R2 * L1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + g.tid;
            if (NW % NT == 0 || w < NW) {
                const int xb = w % L1, ja = (w / L1) % PA::R2, c = w / (L1 * PA::R2);
                stage_smem<PA::R1, false, true>(tile + c * SC + xb * S + ja, PA::R2, tw0, ja);
            }
        }
        gsync<NT>(g);
    }
    plane_middle<LG0, LG1, NCOMP, NT, false>(tile, tw1, g);
    // b stage 2 (no twiddles) -> global; lanes over x0: coalesced
    {
        constexpr int NW = NCOMP * L0 * PB::R1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + g.tid;
            if (NW % NT == 0 || w < NW) {
                const int xa = w % L0, bb = (w / L0) % PB::R1, c = w / (L0 * PB::R1);
                const cplx* p = tile + c * SC + (bb * PB::R2) * S + xa;
                cplx v[PB::R2];
#pragma unroll
                for (int m = 0; m < PB::R2; m++) v[m] = p[m * S];
                bfly<PB::R2, false>(v);
                cplx* gq = field + (long long)c * V + xbase + ((bb * PB::R2) << LG0) + xa;
#pragma unroll
                for (int m = 0; m < PB::R2; m++) st_field(gq + (m << LG0), v[m]);
            }
        }
    }
}

// Sum of two values over a group of NT threads in a fixed order (warp shuffle tree, then warp 0 of the group over the
// warp partials); result valid in group thread 0.  red: 64 doubles of the group's own.  Contains one group barrier.
template <int NT>
__device__ __forceinline__ void group_sum2(double& a, double& b, double* red, const Grp& g) {
    a = warp_sum(a); b = warp_sum(b);
    const int w = g.tid >> 5, l = g.tid & 31;
    constexpr int nw = NT / 32;
    if (l == 0) { red[w] = a; red[32 + w] = b; }
    gsync<NT>(g);
    if (w == 0) {
        a = (l < nw) ? red[l] : 0.0;
        b = (l < nw) ? red[32 + l] : 0.0;
        a = warp_sum(a); b = warp_sum(b);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Pass A, memory phase: S1 of one (x2,x3) plane -> the 4 component tiles, theta/F partial of the plane -> partials.
// Ends with a group barrier (the tile is complete).
template <int LG0, int LG1, int NC, int NT>
__device__ __forceinline__ void pass_a_delta(const cplx* __restrict__ links, const Geom& G, int plane, cplx* __restrict__ tile, double* red,
                                             double2* __restrict__ partials, const Grp& g) {
    constexpr int L0 = 1 << LG0, L1 = 1 << LG1, S = L0 + 1, SC = S * L1, nP = L0 * L1;
    const long long xbase = (long long)plane << (LG0 + LG1);
    double th = 0, fs = 0;
#pragma unroll 1
    for (int e = g.tid; e < nP; e += NT) {
        cplx f0, f1, f2, f3;
        double t_, f_;
#if LGF_FA_PREFETCH_NEXT
        if (e + NT < nP && prefetch_lane()) {   // own links of this thread's next site: DRAM -> L2 while this site is computed
            const cplx* q = links + xbase + e + NT;
#pragma unroll
            for (int k = 0; k < 4 * NC; k++) prefetch_line_l2(q + (long long)k * G.V);
        }
#endif
        delta_site<NC>(links, G, xbase + e, f0, f1, f2, f3, t_, f_);
        th += t_; fs += f_;
        const int o = (e & (L0 - 1)) + (e >> LG0) * S;
        tile[o] = f0; tile[SC + o] = f1; tile[2 * SC + o] = f2; tile[3 * SC + o] = f3;
    }
    group_sum2<NT>(th, fs, red, g);     // its barrier also orders the tile writes
    if (g.tid == 0) partials[plane] = make_double2(th, fs);
    gsync<NT>(g);
}

// S5 by one whole CTA (all its threads call this): sums the partials in the order k_finalize uses (strided per thread,
// then the fixed tree: bit-identical), writes F, theta and the history and raises the stop flag.
// FinArgs::on = number of partials the first CTA of pass B has to reduce (0: k_finalize already did it).
struct FinArgs { double2* hist; double inv3V, inv12V; int on; };
template <int NT>
__device__ __forceinline__ void finalize_cta(const double2* partials, int n, Ctl* ctl, const FinArgs& fa, double* red) {
    double a = 0, b = 0;
    for (int i = threadIdx.x; i < n; i += NT) { const double2 p = __ldcg(partials + i); a += p.x; b += p.y; }
    block_sum2(a, b, red);
    if (threadIdx.x == 0) {
        s5_decide(ctl, fa.hist, a * fa.inv3V, b * fa.inv12V);
    }
    __syncthreads();
}
// S5 inside pass B: the partials of pass A are complete when pass B starts, so its CTA 0 does
// the reduction and the stop decision before its own tile -- no k_finalize launch, no fence.  Pass B itself never needs
// the decision (it only transforms the scratch field; a CTA that already sees the flag may skip its tile, which nobody
// reads once the flag is up); pass C and the update start after this kernel has ended and see it.
// Entry of the pass-B kernels.  With S5 inside pass B the stop flag can be raised by CTA 0 WHILE other CTAs of the same
// kernel start, so a CTA must take ONE reading of it: thread 0 reads it at entry into shared memory, and the CTA acts on
// it only behind its first regular barrier (PASS_B_EXIT_IF_DONE) -- if every thread read the flag for itself the warps
// of a CTA could disagree and the CTA would hang at its next barrier, and a barrier of its own right behind
// griddepcontrol.wait costs 60 us per iteration under programmatic dependent launch (measured).  What a CTA does before
// that barrier only touches its shared-memory tile.  CTA 0 alone synchronises at once, because it has to know whether the
// run is already over before it reduces the partials of the S1 that has just run (fa.on of them; 0: k_finalize did it).
template <int NT>
__device__ __forceinline__ void pass_b_entry(const double2* partials, const FinArgs& fa, Ctl* ctl, int* s_done) {
    __shared__ double red_fin[64];
    // Every thread reads one word of the control block right behind griddepcontrol.wait and branches on it (hist_cap
    // never changes while kernels run and is never negative).  Measured: without such a read the first instructions
    // behind the wait are the field loads of phase 1 and the iteration takes 373 us under programmatic dependent
    // launch; with it 310 us -- as with the per-thread "if (ctl->done) return" of the other kernels.
    if (ctl->hist_cap < 0) return;
    if (threadIdx.x == 0) *s_done = __ldcg(&ctl->done);
    if (fa.on > 0 && blockIdx.x == 0) {
        __syncthreads();
        if (!*s_done) finalize_cta<NT>(partials, fa.on, ctl, fa, red_fin);
    }
}

// Pass A: S1 (Delta, theta/F partials) + forward FFT over axes 0,1 of one (x2,x3) plane, all 4 components.
template <int LG0, int LG1, int NC, int NT>
__global__ void __launch_bounds__(NT, LGF_FA_MINB_DELTA) k_fa_delta_fwd(const cplx* __restrict__ links, cplx* __restrict__ field, double2* __restrict__ partials,
                                                     Geom G, FftTables T, const Ctl* __restrict__ ctl) {
    pdl_enter();
    if (ctl->done) return;
    constexpr int L0 = 1 << LG0, L1 = 1 << LG1, S = L0 + 1, SC = S * L1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw0 = tile + 4 * SC;
    cplx* tw1 = tw0 + L0;
    __shared__ double red[64];
    const Grp g{(int)threadIdx.x, 0};
    for (int i = threadIdx.x; i < L0; i += NT) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += NT) tw1[i] = T.tw[1][i];
    // planes from the last one down: the link update before this kernel walks upwards and leaves its last planes in L2
    const int plane = (int)gridDim.x - 1 - (int)blockIdx.x;
    pass_a_delta<LG0, LG1, NC, NT>(links, G, plane, tile, red, partials, g);
    plane_forward_store<LG0, LG1, NT>(tile, tw0, tw1, field, G.V, (long long)plane << (LG0 + LG1), g);
}

// Pass A for 64 x 64 planes on a CTA PAIR (thread-block cluster of 2, distributed shared memory): the four component
// tiles (266 KB) do not fit one SM, so CTA r of the pair keeps components 2r, 2r+1 (133 KB).  Each CTA computes S1 for
// half of the plane's rows -- all four components of a site come out of the same eight links -- and writes the two
// components its partner owns straight into the partner's tile (st.shared::cluster through map_shared_rank).  After
// one cluster barrier each CTA transforms its two components.  S1 stays fused (no Delta round trip through HBM:
// 1536 instead of 1664 B/site) and the links are still read once.  Two (theta, F) partials per plane.
template <int LG0, int LG1, int NC, int NT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NT, 1)
k_cl_delta_fwd(const cplx* __restrict__ links, cplx* __restrict__ field, double2* __restrict__ partials, Geom G, FftTables T,
               const Ctl* __restrict__ ctl) {
    pdl_enter();
    if (ctl->done) return;                               // uniform over the grid: both CTAs of a pair leave together
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    constexpr int L0 = 1 << LG0, L1 = 1 << LG1, S = L0 + 1, SC = S * L1, nP = L0 * L1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);      // [2][L1][S]
    cplx* tw0 = tile + 2 * SC;
    cplx* tw1 = tw0 + L0;
    __shared__ double red[64];
    const int r = (int)cluster.block_rank();             // which half of the rows, which pair of components
    cplx* peer = cluster.map_shared_rank(tile, r ^ 1);
    // The planes are walked in x2 bands of 16: x2 fastest inside a band, then x3, then the bands.  The backward neighbours
    // U_2(x-2) and U_3(x-3) live in the planes (x2-1, x3) and (x2, x3-1); in plain order the latter was read 64 planes =
    // 100 MB of links earlier and has left L2 (ncu at 64^4: 7.90 GB of DRAM reads against 6.44 GB of links), here 16.
    int plane = (int)(gridDim.x >> 1) - 1 - (int)(blockIdx.x >> 1);      // from the last plane down (see k_fa_delta_fwd)
    if (G.L[2] >= 32) {
        const int x2l = plane & 15, x3 = (plane >> 4) & (G.L[3] - 1), bnd = plane >> (4 + G.lg[3]);
        plane = (bnd * 16 + x2l) + (x3 << G.lg[2]);
    }
    const long long xbase = (long long)plane << (LG0 + LG1);
    const Grp g{(int)threadIdx.x, 0};
    for (int i = threadIdx.x; i < L0; i += NT) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += NT) tw1[i] = T.tw[1][i];
    double th = 0, fs = 0;
#pragma unroll 1
    for (int e = r * (nP / 2) + threadIdx.x; e < (r + 1) * (nP / 2); e += NT) {
        cplx f[4];
        double t_, f_;
        delta_site<NC>(links, G, xbase + e, f[0], f[1], f[2], f[3], t_, f_);
        th += t_; fs += f_;
        const int o = (e & (L0 - 1)) + (e >> LG0) * S;
        cplx* own = tile + o;
        cplx* oth = peer + o;
        if (r == 0) { own[0] = f[0]; own[SC] = f[1]; oth[0] = f[2]; oth[SC] = f[3]; }
        else { oth[0] = f[0]; oth[SC] = f[1]; own[0] = f[2]; own[SC] = f[3]; }
    }
    block_sum2(th, fs, red);
    if (threadIdx.x == 0) partials[2 * plane + r] = make_double2(th, fs);
    cluster.sync();                                      // both halves of both tiles are in place (release/acquire)
    plane_forward_store<LG0, LG1, NT, 2>(tile, tw0, tw1, field + (long long)(2 * r) * G.V, G.V, xbase, g);
}

// Pass A without S1, for planes whose four component tiles do not fit one SM (64 x 64, 32 x 64): forward FFT over axes
// 0,1 of NCOMP components of one plane, Delta read from field (written by k_delta).  blockIdx.x = plane * (4/NCOMP) + group.
template <int LG0, int LG1, int NCOMP, int NT>
__global__ void __launch_bounds__(NT, 2) k_fa_fwd(cplx* __restrict__ field, Geom G, FftTables T, const Ctl* __restrict__ ctl) {
    pdl_enter();
    if (ctl->done) return;
    constexpr int L0 = 1 << LG0, L1 = 1 << LG1, S = L0 + 1, SC = S * L1, nP = L0 * L1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw0 = tile + NCOMP * SC;
    cplx* tw1 = tw0 + L0;
    constexpr int NG = 4 / NCOMP;
    const long long xbase = (long long)(blockIdx.x / NG) << (LG0 + LG1);
    cplx* fbase = field + (long long)((blockIdx.x % NG) * NCOMP) * G.V;
    const Grp g{(int)threadIdx.x, 0};
    for (int i = threadIdx.x; i < L0; i += NT) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += NT) tw1[i] = T.tw[1][i];
#pragma unroll 4
    for (int e = threadIdx.x; e < NCOMP * nP; e += NT) {
        const int c = e >> (LG0 + LG1), r = e & (nP - 1);
        tile[c * SC + (r & (L0 - 1)) + (r >> LG0) * S] = ld_field(fbase + (long long)c * G.V + xbase + r);
    }
    __syncthreads();
    plane_forward_store<LG0, LG1, NT, NCOMP>(tile, tw0, tw1, fbase, G.V, xbase, g);
}

// ---------------------------------------------------------------------------------------------------------------
// Pass C, memory phase: X~ of one plane (NCOMP components from fbase) -> inverse b stage 2 (no twiddles) -> tile.
// Ends with a group barrier.
template <int LG0, int LG1, int NCOMP, int NT>
__device__ __forceinline__ void pass_c_load(const cplx* __restrict__ fbase, long long V, cplx* __restrict__ tile, const Grp& g) {
    using PB = Plan2<LG1, true>;
    constexpr int L0 = 1 << LG0, L1 = 1 << LG1, S = L0 + 1, SC = S * L1;
    constexpr int NW = NCOMP * L0 * PB::R1;
#pragma unroll
    for (int w0 = 0; w0 < NW; w0 += NT) {
        const int w = w0 + g.tid;
        if (NW % NT == 0 || w < NW) {
            const int xa = w % L0, bb = (w / L0) % PB::R1, c = w / (L0 * PB::R1);
            const cplx* gq = fbase + (long long)c * V + ((bb * PB::R2) << LG0) + xa;
            cplx v[PB::R2];
#pragma unroll
            for (int m = 0; m < PB::R2; m++) v[m] = ld_field(gq + (m << LG0));
            bfly<PB::R2, true>(v);
            cplx* p = tile + c * SC + (bb * PB::R2) * S + xa;
#pragma unroll
            for (int m = 0; m < PB::R2; m++) p[m * S] = v[m];
        }
    }
    gsync<NT>(g);
}

// Pass C, on-chip phase: the remaining inverse stages of axes 1,0; X -> field (in place), or with WRITE_G the pass ends
// in S3, g(x) = GramSchmidt(1 + (alpha/2) X(x)), rows 0,1 written to gbuf (6 V-arrays) at gbase = gbuf + xbase.
template <int LG0, int LG1, int NCOMP, int NT, bool WRITE_G>
__device__ __forceinline__ void pass_c_finish(cplx* __restrict__ fbase, cplx* __restrict__ gbase, double half_alpha, long long V, cplx* __restrict__ tile,
                                              const cplx* __restrict__ tw0, const cplx* __restrict__ tw1, const Grp& g) {
    using PA = Plan2<LG0, false>;
    using PB = Plan2<LG1, true>;
    constexpr int L0 = PA::L, L1 = PB::L, S = L0 + 1, SC = S * L1;
    plane_middle<LG0, LG1, NCOMP, NT, true>(tile, tw1, g);
    if constexpr (WRITE_G) {
        // a stage 1 inverse in place (lanes over rows: odd stride, conflict-free), then S3 per site
        constexpr int NW = NCOMP * PA::R2 * L1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + g.tid;
            if (NW % NT == 0 || w < NW) {
                const int xb = w % L1, ja = (w / L1) % PA::R2, c = w / (L1 * PA::R2);
                stage_smem<PA::R1, true, true>(tile + c * SC + xb * S + ja, PA::R2, tw0, ja);
            }
        }
        gsync<NT>(g);
        constexpr int nP = L0 * L1;
#pragma unroll 1
        for (int e = g.tid; e < nP; e += NT) {
            const int o = (e & (L0 - 1)) + (e >> LG0) * S;
            cplx gm[9];
            build_g(tile[o], tile[SC + o], tile[2 * SC + o], tile[3 * SC + o], (real)half_alpha, gm);
#pragma unroll
            for (int c = 0; c < 6; c++) gbase[(long long)c * V + e] = gm[c];
        }
    } else {
        // a stage 1 inverse (twiddles conj tw0[k ja]) -> global.  Lane order (R2 = 4): a quarter-warp is 4 consecutive ja
        // (one 64 B segment) of two rows 4 apart: its shared-memory reads are conflict-free (16-byte bank group =
        // (xb + ja + 4m) mod 8 with the odd row stride) and its global store touches 2 lines, 8 per warp instruction.
        // (Lanes over 8 rows first, as in the first version, made every quarter-warp touch 8 lines: ncu showed the pass
        // bound by L1TEX data-pipe wavefronts, 32.7 k global per SM against 10.6 k now.)  R2 = 8: 128 B per quarter-warp.
        constexpr int NW = NCOMP * PA::R2 * L1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + g.tid;
            if (NW % NT == 0 || w < NW) {
                int ja, xb;
                if constexpr (PA::R2 >= 8) { ja = w % PA::R2; xb = (w / PA::R2) % L1; }
                else {
                    static_assert(PA::R2 == 4, "lane order below");
                    const int t = w >> 2;
                    ja = w & 3; xb = (((t >> 1) & 3) | ((t & 1) << 2)) + 8 * ((t >> 3) % (L1 / 8));
                }
                const int c = w / (PA::R2 * L1);
                const cplx* p = tile + c * SC + xb * S + ja;
                cplx v[PA::R1];
#pragma unroll
                for (int m = 0; m < PA::R1; m++) v[m] = p[m * PA::R2];
                stage_regs<PA::R1, true, true>(v, tw0, ja);
                cplx* gq = fbase + (long long)c * V + (xb << LG0) + ja;
#pragma unroll
                for (int m = 0; m < PA::R1; m++) st_field(gq + m * PA::R2, v[m]);
            }
        }
    }
}

// Pass C: inverse FFT over axes 1,0 of one (x2,x3) plane for NCOMP components (blockIdx.x = plane * (4/NCOMP) + group).
template <int LG0, int LG1, int NCOMP, int NT, bool WRITE_G>
__global__ void __launch_bounds__(NT, LGF_FA_MINB_INV) k_fa_inv(cplx* __restrict__ field, cplx* __restrict__ gbuf, double half_alpha, Geom G, FftTables T,
                                                                const Ctl* __restrict__ ctl) {
    static_assert(!WRITE_G || NCOMP == 4, "g needs all four components of X");
    pdl_enter();
    if (ctl->done) return;
    constexpr int L0 = 1 << LG0, L1 = 1 << LG1, S = L0 + 1, SC = S * L1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw0 = tile + NCOMP * SC;
    cplx* tw1 = tw0 + L0;
    constexpr int NG = 4 / NCOMP;
    const long long xbase = (long long)(blockIdx.x / NG) << (LG0 + LG1);
    cplx* fbase = field + (long long)((blockIdx.x % NG) * NCOMP) * G.V + xbase;
    const Grp g{(int)threadIdx.x, 0};
    for (int i = threadIdx.x; i < L0; i += NT) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += NT) tw1[i] = T.tw[1][i];
    pass_c_load<LG0, LG1, NCOMP, NT>(fbase, G.V, tile, g);      // its barrier also publishes the twiddles
    pass_c_finish<LG0, LG1, NCOMP, NT, WRITE_G>(fbase, WRITE_G ? gbuf + xbase : nullptr, half_alpha, G.V, tile, tw0, tw1, g);
}

// ---------------------------------------------------------------------------------------------------------------
// Pass B works on the (x2,x3) extent of one (component, x1, chunk of C0 = 2^LGC consecutive x0):
// tile[i3][i2][i0], S1 = C0, S2 = C0*L2 (+C0 when C0 < 8: keeps quarter-warps conflict-free).
// Work item index = chunk + nChunks*(x1 + L1*comp).
template <int LG2, int LGC> struct MidGeom {
    static constexpr int L2 = 1 << LG2, C0 = 1 << LGC, S1 = C0, S2 = C0 * L2 + (C0 < 8 ? C0 : 0);
};
struct MidItem {
    cplx* gp;        // field + comp*V + chunk*C0 + x1*L0 + i0
    double s01;      // s[0][x0] + s[1][x1] of this thread's x0
};
template <int LGC>
__device__ __forceinline__ MidItem mid_item(cplx* __restrict__ field, const Geom& G, const FftTables& T, int item, int i0) {
    const int lgChunks = G.lg[0] - LGC;
    const int chunk = item & ((1 << lgChunks) - 1);
    const int x1 = (item >> lgChunks) & (G.L[1] - 1);
    const int comp = item >> (lgChunks + G.lg[1]);
    MidItem it;
    it.gp = field + (long long)comp * G.V + (chunk << LGC) + ((long long)x1 << G.sh[1]) + i0;
    it.s01 = T.s[0][(chunk << LGC) + i0] + T.s[1][x1];
    return it;
}

// Pass B, memory phase: global -> axis-2 stage 1 (points i2 = ja + m R2, twiddles tw2[k ja]) -> tile.  Ends with a
// group barrier.  tl = tile + i0.
template <int LG2, int LG3, int LGC, int NT>
__device__ __forceinline__ void pass_b_load(const cplx* __restrict__ gp, int sh2, int sh3, cplx* __restrict__ tl, const cplx* __restrict__ tw2, const Grp& g) {
    using PA = PlanM<LG2, false>;
    using PB = PlanM<LG3, true>;
    using MG = MidGeom<LG2, LGC>;
    constexpr int L3 = PB::L, C0 = MG::C0, S1 = MG::S1, S2 = MG::S2;
    constexpr int NW = C0 * PA::R2 * L3;
#pragma unroll
    for (int w0 = 0; w0 < NW; w0 += NT) {
        const int w = w0 + g.tid;
        if (NW % NT == 0 || w < NW) {
            const int ja = (w / C0) % PA::R2, i3 = w / (C0 * PA::R2);
            const cplx* gq = gp + ((long long)ja << sh2) + ((long long)i3 << sh3);
            cplx v[PA::R1];
#pragma unroll
            for (int m = 0; m < PA::R1; m++) v[m] = ld_field(gq + ((long long)(m * PA::R2) << sh2));
            stage_regs<PA::R1, false, true>(v, tw2, ja);
            cplx* p = tl + ja * S1 + i3 * S2;
#pragma unroll
            for (int m = 0; m < PA::R1; m++) p[m * PA::R2 * S1] = v[m];
        }
    }
    gsync<NT>(g);
}

// Pass B, on-chip phase: the remaining forward stages, the p2max/p2 filter, the inverse stages, last one -> global.
template <int LG2, int LG3, int LGC, int NT>
__device__ __forceinline__ void pass_b_finish(cplx* __restrict__ gp, double s01, int sh2, int sh3, double scale, cplx* __restrict__ tl,
                                              const cplx* __restrict__ tw2, const cplx* __restrict__ tw3, const double* __restrict__ s2,
                                              const double* __restrict__ s3, const Grp& g) {
    using PA = PlanM<LG2, false>;
    using PB = PlanM<LG3, true>;
    using MG = MidGeom<LG2, LGC>;
    constexpr int L2 = PA::L, L3 = PB::L, C0 = MG::C0, S1 = MG::S1, S2 = MG::S2;
    // middle stages, forward and (after the filter) inverse
    auto middle = [&](auto inv_tag) {
        constexpr bool INV = decltype(inv_tag)::value;
        if constexpr (PA::R2 * PB::R1 <= 16) {
            constexpr int NW = C0 * PB::R2 * PA::R1;
#pragma unroll
            for (int w0 = 0; w0 < NW; w0 += NT) {
                const int w = w0 + g.tid;
                if (NW % NT == 0 || w < NW) {
                    const int jb = (w / C0) % PB::R2, ba = w / (C0 * PB::R2);
                    block_smem<PA::R2, PB::R1, INV>(tl + ba * PA::R2 * S1 + jb * S2, S1, PB::R2 * S2, tw3, jb);
                }
            }
            gsync<NT>(g);
        } else {
            auto a2 = [&]() {
                constexpr int NW = C0 * PA::R1 * L3;
#pragma unroll
                for (int w0 = 0; w0 < NW; w0 += NT) {
                    const int w = w0 + g.tid;
                    if (NW % NT == 0 || w < NW) {
                        const int ba = (w / C0) % PA::R1, i3 = w / (C0 * PA::R1);
                        stage_smem<PA::R2, INV, false>(tl + ba * PA::R2 * S1 + i3 * S2, S1, nullptr, 0);
                    }
                }
                gsync<NT>(g);
            };
            auto b1 = [&]() {
                constexpr int NW = C0 * L2 * PB::R2;
#pragma unroll
                for (int w0 = 0; w0 < NW; w0 += NT) {
                    const int w = w0 + g.tid;
                    if (NW % NT == 0 || w < NW) {
                        const int i2 = (w / C0) % L2, jb = w / (C0 * L2);
                        stage_smem<PB::R1, INV, true>(tl + i2 * S1 + jb * S2, PB::R2 * S2, tw3, jb);
                    }
                }
                gsync<NT>(g);
            };
            if constexpr (INV) { b1(); a2(); } else { a2(); b1(); }
        }
    };
    middle(std::false_type{});
    // axis-3 stage 2 forward, S2b filter X~ = (16 / (V p2)) Delta~ at the stored positions (zero mode -> 0), axis-3
    // stage 2 inverse, all on the same registers                                             [north_star step 2]
    {
        constexpr int NW = C0 * L2 * PB::R1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + g.tid;
            if (NW % NT == 0 || w < NW) {
                const int i2 = (w / C0) % L2, bb = w / (C0 * L2);
                cplx* p = tl + i2 * S1 + (bb * PB::R2) * S2;
                cplx v[PB::R2];
#pragma unroll
                for (int m = 0; m < PB::R2; m++) v[m] = p[m * S2];
                bfly<PB::R2, false>(v);
                const double s012 = s01 + s2[i2];
#pragma unroll
                for (int m = 0; m < PB::R2; m++) {
                    const double p2 = s012 + s3[bb * PB::R2 + m];
                    const double wgt = filter_weight(scale, p2);
                    v[m] = cscale(v[m], (real)wgt);
                }
                bfly<PB::R2, true>(v);
#pragma unroll
                for (int m = 0; m < PB::R2; m++) p[m * S2] = v[m];
            }
        }
        gsync<NT>(g);
    }
    middle(std::true_type{});
    // tile -> axis-2 stage 1 inverse -> global
    {
        constexpr int NW = C0 * PA::R2 * L3;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + g.tid;
            if (NW % NT == 0 || w < NW) {
                const int ja = (w / C0) % PA::R2, i3 = w / (C0 * PA::R2);
                const cplx* p = tl + ja * S1 + i3 * S2;
                cplx v[PA::R1];
#pragma unroll
                for (int m = 0; m < PA::R1; m++) v[m] = p[m * PA::R2 * S1];
                stage_regs<PA::R1, true, true>(v, tw2, ja);
                cplx* gq = gp + ((long long)ja << sh2) + ((long long)i3 << sh3);
#pragma unroll
                for (int m = 0; m < PA::R1; m++) st_field(gq + ((long long)(m * PA::R2) << sh2), v[m]);
            }
        }
    }
}

// Pass B: forward over axes 2,3, filter, inverse over axes 3,2, one work item per CTA.
template <int LG2, int LG3, int LGC, int NT>
__global__ void __launch_bounds__(NT, (NT > 256) ? 1 : LGF_FA_MINB_MID) k_fa_mid(cplx* __restrict__ field, Geom G, FftTables T, double scale, Ctl* ctl, const double2* partials, FinArgs fa) {
    pdl_enter();
    __shared__ int s_done;
    pass_b_entry<NT>(partials, fa, ctl, &s_done);
    using MG = MidGeom<LG2, LGC>;
    constexpr int L2 = 1 << LG2, L3 = 1 << LG3, C0 = MG::C0;
    static_assert(NT % C0 == 0, "a thread keeps its x0 offset");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw2 = tile + MG::S2 * L3;
    cplx* tw3 = tw2 + L2;
    double* s2 = reinterpret_cast<double*>(tw3 + L3);
    double* s3 = s2 + L2;
    const Grp g{(int)threadIdx.x, 0};
    const int i0 = threadIdx.x % C0;
    const MidItem it = mid_item<LGC>(field, G, T, blockIdx.x, i0);
    for (int i = threadIdx.x; i < L2; i += NT) { tw2[i] = T.tw[2][i]; s2[i] = T.s[2][i]; }
    for (int i = threadIdx.x; i < L3; i += NT) { tw3[i] = T.tw[3][i]; s3[i] = T.s[3][i]; }
    __syncthreads();
    if (s_done) return;                                  // one reading per CTA, behind a barrier (pass_b_entry)
    pass_b_load<LG2, LG3, LGC, NT>(it.gp, G.sh[2], G.sh[3], tile + i0, tw2, g);
    pass_b_finish<LG2, LG3, LGC, NT>(it.gp, it.s01, G.sh[2], G.sh[3], scale, tile + i0, tw2, tw3, s2, s3, g);
}


// ---------------------------------------------------------------------------------------------------------------
// Pass B with whole lines in registers (extents 16 and 32).  A thread takes one line of the tile at a time and runs
// the complete forward (or inverse) transform of that axis on it in registers -- same stages, radices and stored
// order as the passes above (Plan2), twiddles from constant-memory tables with compile-time indices, so they are
// instruction operands, not loads.  Per point the tile is written twice and read twice (the stage-wise pass B: four
// times each) and the pass has two barriers instead of five.
//   phase 1: axis-2 lines straight from global memory -> forward -> tile
//   phase 2: axis-3 lines: forward, p2max/p2 filter, inverse, in place
//   phase 3: axis-2 lines: inverse -> straight to global memory
__constant__ real c_tw16[16][2] = {      // exp(-2 pi i k / 16), correctly rounded
    {(real)1.0, (real)-0.0}, {(real)0.9238795325112867, (real)-0.3826834323650898},
    {(real)0.7071067811865476, (real)-0.7071067811865476}, {(real)0.3826834323650898, (real)-0.9238795325112867},
    {(real)0.0, (real)-1.0}, {(real)-0.3826834323650898, (real)-0.9238795325112867},
    {(real)-0.7071067811865476, (real)-0.7071067811865476}, {(real)-0.9238795325112867, (real)-0.3826834323650898},
    {(real)-1.0, (real)-0.0}, {(real)-0.9238795325112867, (real)0.3826834323650898},
    {(real)-0.7071067811865476, (real)0.7071067811865476}, {(real)-0.3826834323650898, (real)0.9238795325112867},
    {(real)0.0, (real)1.0}, {(real)0.3826834323650898, (real)0.9238795325112867},
    {(real)0.7071067811865476, (real)0.7071067811865476}, {(real)0.9238795325112867, (real)0.3826834323650898},
};
__constant__ real c_tw32[32][2] = {      // exp(-2 pi i k / 32), correctly rounded
    {(real)1.0, (real)-0.0}, {(real)0.9807852804032304, (real)-0.19509032201612828},
    {(real)0.9238795325112867, (real)-0.3826834323650898}, {(real)0.8314696123025452, (real)-0.5555702330196022},
    {(real)0.7071067811865476, (real)-0.7071067811865476}, {(real)0.5555702330196022, (real)-0.8314696123025452},
    {(real)0.3826834323650898, (real)-0.9238795325112867}, {(real)0.19509032201612828, (real)-0.9807852804032304},
    {(real)0.0, (real)-1.0}, {(real)-0.19509032201612828, (real)-0.9807852804032304},
    {(real)-0.3826834323650898, (real)-0.9238795325112867}, {(real)-0.5555702330196022, (real)-0.8314696123025452},
    {(real)-0.7071067811865476, (real)-0.7071067811865476}, {(real)-0.8314696123025452, (real)-0.5555702330196022},
    {(real)-0.9238795325112867, (real)-0.3826834323650898}, {(real)-0.9807852804032304, (real)-0.19509032201612828},
    {(real)-1.0, (real)-0.0}, {(real)-0.9807852804032304, (real)0.19509032201612828},
    {(real)-0.9238795325112867, (real)0.3826834323650898}, {(real)-0.8314696123025452, (real)0.5555702330196022},
    {(real)-0.7071067811865476, (real)0.7071067811865476}, {(real)-0.5555702330196022, (real)0.8314696123025452},
    {(real)-0.3826834323650898, (real)0.9238795325112867}, {(real)-0.19509032201612828, (real)0.9807852804032304},
    {(real)0.0, (real)1.0}, {(real)0.19509032201612828, (real)0.9807852804032304},
    {(real)0.3826834323650898, (real)0.9238795325112867}, {(real)0.5555702330196022, (real)0.8314696123025452},
    {(real)0.7071067811865476, (real)0.7071067811865476}, {(real)0.8314696123025452, (real)0.5555702330196022},
    {(real)0.9238795325112867, (real)0.3826834323650898}, {(real)0.9807852804032304, (real)0.19509032201612828},
};
template <int LG> __device__ __forceinline__ cplx ctw(int k) {      // k is a compile-time constant after unrolling
    if constexpr (LG == 4) return mk(c_tw16[k][0], c_tw16[k][1]);
    else return mk(c_tw32[k][0], c_tw32[k][1]);
}

// Complete transform of one line of L = R1 R2 points in registers: the two stages of Plan2<LG, B>, in place, stored
// (digit-reversed) order out of the forward transform and into the inverse one.
template <int LG, bool B, bool INV>
__device__ __forceinline__ void line_fft(cplx (&v)[1 << LG]) {
    using P = Plan2<LG, B>;
    auto stage1 = [&]() {        // points ja + m R2, twiddles W_L^{k ja}
#pragma unroll
        for (int ja = 0; ja < P::R2; ja++) {
            cplx x[P::R1];
#pragma unroll
            for (int m = 0; m < P::R1; m++) x[m] = v[ja + m * P::R2];
            if constexpr (INV) {
#pragma unroll
                for (int k = 1; k < P::R1; k++) if (ja) x[k] = cmulc(x[k], ctw<LG>(k * ja));
                bfly<P::R1, true>(x);
            } else {
                bfly<P::R1, false>(x);
#pragma unroll
                for (int k = 1; k < P::R1; k++) if (ja) x[k] = cmul(x[k], ctw<LG>(k * ja));
            }
#pragma unroll
            for (int m = 0; m < P::R1; m++) v[ja + m * P::R2] = x[m];
        }
    };
    auto stage2 = [&]() {        // contiguous sub-blocks of R2 points, unit twiddles
#pragma unroll
        for (int ba = 0; ba < P::R1; ba++) {
            cplx x[P::R2];
#pragma unroll
            for (int m = 0; m < P::R2; m++) x[m] = v[ba * P::R2 + m];
            bfly<P::R2, INV>(x);
#pragma unroll
            for (int m = 0; m < P::R2; m++) v[ba * P::R2 + m] = x[m];
        }
    };
    if constexpr (INV) { stage2(); stage1(); } else { stage1(); stage2(); }
}

#ifndef LGF_FR_NT
#define LGF_FR_NT 128
#endif
#ifndef LGF_FR_MINB
#define LGF_FR_MINB 2
#endif
template <int LG2, int LG3, int LGC, int NT, bool COULOMB = false>
__global__ void __launch_bounds__(NT, LGF_FR_MINB) k_fr_mid(cplx* __restrict__ field, Geom G, FftTables T, double scale, Ctl* ctl, const double2* partials, FinArgs fa) {
    pdl_enter();
    __shared__ int s_done;
    pass_b_entry<NT>(partials, fa, ctl, &s_done);
    using MG = MidGeom<LG2, LGC>;
    constexpr int L2 = 1 << LG2, L3 = 1 << LG3, C0 = MG::C0, S1 = MG::S1, S2 = MG::S2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    double* s2 = reinterpret_cast<double*>(tile + S2 * L3);
    double* s3 = s2 + L2;
    for (int i = threadIdx.x; i < L2; i += NT) s2[i] = T.s[2][i];
    for (int i = threadIdx.x; i < L3; i += NT) s3[i] = T.s[3][i];
    const int lgChunks = G.lg[0] - LGC;
    const int chunk = blockIdx.x & ((1 << lgChunks) - 1);
    const int x1 = (blockIdx.x >> lgChunks) & (G.L[1] - 1);
    const int comp = blockIdx.x >> (lgChunks + G.lg[1]);
    cplx* gbase = field + (long long)comp * G.V + (chunk << LGC) + ((long long)x1 << G.sh[1]);
    const int sh2 = G.sh[2], sh3 = G.sh[3];
    if constexpr (COULOMB) {
        // Coulomb gauge: the filter does not depend on the axis-3 momentum, so the transform pair along axis 3 cancels and
        // every axis-2 line is finished on its own: forward, filter, inverse in registers, no shared memory, no barrier
        __syncthreads();                                     // s2 is complete
        if (s_done) return;
#pragma unroll 1
        for (int ln = threadIdx.x; ln < C0 * L3; ln += NT) {
            const int i0 = ln % C0, i3 = ln / C0;
            cplx* gq = gbase + i0 + ((long long)i3 << sh3);
            cplx v[L2];
#pragma unroll
            for (int m = 0; m < L2; m++) v[m] = ld_field(gq + ((long long)m << sh2));
            line_fft<LG2, false, false>(v);
            const double s01 = T.s[0][(chunk << LGC) + i0] + T.s[1][x1];
#pragma unroll
            for (int m = 0; m < L2; m++) {
                const double p2 = s01 + s2[m];
                v[m] = cscale(v[m], (real)filter_weight(scale * (double)L3, p2));      // no 1/L3: axis 3 is not transformed
            }
            line_fft<LG2, false, true>(v);
#pragma unroll
            for (int m = 0; m < L2; m++) st_field(gq + ((long long)m << sh2), v[m]);
        }
        return;
    }
    // phase 1: lines along axis 2, one per (i0, i3)
#pragma unroll 1
    for (int ln = threadIdx.x; ln < C0 * L3; ln += NT) {
        const int i0 = ln % C0, i3 = ln / C0;
        const cplx* gq = gbase + i0 + ((long long)i3 << sh3);
        cplx v[L2];
#pragma unroll
        for (int m = 0; m < L2; m++) v[m] = ld_field(gq + ((long long)m << sh2));
        line_fft<LG2, false, false>(v);
        cplx* p = tile + i0 + i3 * S2;
#pragma unroll
        for (int m = 0; m < L2; m++) p[m * S1] = v[m];
    }
    __syncthreads();
    if (s_done) return;                                  // one reading per CTA, behind a barrier (pass_b_entry)
    // phase 2: lines along axis 3, one per (i0, i2): forward, filter X~ = (p2max / (V p2)) Delta~ at the stored positions
    // (zero mode -> 0), inverse                                                                  [north_star step 2]
#pragma unroll 1
    for (int ln = threadIdx.x; ln < C0 * L2; ln += NT) {
        const int i0 = ln % C0, i2 = ln / C0;
        cplx* p = tile + i0 + i2 * S1;
        cplx v[L3];
#pragma unroll
        for (int m = 0; m < L3; m++) v[m] = p[m * S2];
        line_fft<LG3, true, false>(v);
        const double s012 = T.s[0][(chunk << LGC) + i0] + T.s[1][x1] + s2[i2];
#pragma unroll
        for (int m = 0; m < L3; m++) {
            const double p2 = s012 + s3[m];
            v[m] = cscale(v[m], (real)filter_weight(scale, p2));
        }
        line_fft<LG3, true, true>(v);
#pragma unroll
        for (int m = 0; m < L3; m++) p[m * S2] = v[m];
    }
    __syncthreads();
    // phase 3: lines along axis 2 again: inverse, straight to global memory
#pragma unroll 1
    for (int ln = threadIdx.x; ln < C0 * L3; ln += NT) {
        const int i0 = ln % C0, i3 = ln / C0;
        const cplx* p = tile + i0 + i3 * S2;
        cplx v[L2];
#pragma unroll
        for (int m = 0; m < L2; m++) v[m] = p[m * S1];
        line_fft<LG2, false, true>(v);
        cplx* gq = gbase + i0 + ((long long)i3 << sh3);
#pragma unroll
        for (int m = 0; m < L2; m++) st_field(gq + ((long long)m << sh2), v[m]);
    }
}

}  // namespace lgf
