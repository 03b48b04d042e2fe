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
#include "kernels.cuh"

// resident CTAs per SM the passes are compiled for (register cap = 65536 / (NT * MINB)).  Measured on B200 at 32^4
// (CUDA events per launch): pass A 118.9 us at 1 CTA/SM, 107.7 at 2, 143.2 at 3 (spills); pass B 66.0 / 47.3 / 59.3.
#ifndef LGF_FA_MINB_DELTA
#define LGF_FA_MINB_DELTA 2
#endif
#ifndef LGF_FA_MINB_MID
#define LGF_FA_MINB_MID 2
#endif
#ifndef LGF_FA_MINB_INV
#define LGF_FA_MINB_INV 1
#endif

namespace lgf {

// Two-stage plan of an axis of length 2^LG (LG = 4, 5, 6); B = axis 1 or 3.  Must agree with make_plan().
template <int LG, bool B> struct Plan2 {
    static_assert(LG >= 4 && LG <= 6, "fast FFT passes cover L = 16, 32, 64");
    static constexpr int LG1 = (LG == 4) ? 2 : ((LG == 5) ? (B ? 2 : 3) : 3);
    static constexpr int LG2 = LG - LG1;
    static constexpr int R1 = 1 << LG1, R2 = 1 << LG2, L = 1 << LG;
};

// Forward stage on registers: y = DFT_R(v), then y_k *= tw[k*t]  (t = j * L/N: W_N^{jk} = tw[k t]).
// Inverse stage: v_k *= conj(tw[k t]), then y = IDFT_R(v).
template <int R, bool INV, bool TW>
__device__ __forceinline__ void stage_regs(cplx (&v)[R], const cplx* __restrict__ tw, int t) {
    if constexpr (INV) {
        if constexpr (TW) {
#pragma unroll
            for (int k = 1; k < R; k++) v[k] = cmulc(v[k], tw[k * t]);
        }
        bfly<R, true>(v);
    } else {
        bfly<R, false>(v);
        if constexpr (TW) {
#pragma unroll
            for (int k = 1; k < R; k++) v[k] = cmul(v[k], tw[k * t]);
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
// Ends with __syncthreads().
template <int LGA, int LGB, int NCOMP, int NT, bool INV>
__device__ __forceinline__ void plane_middle(cplx* __restrict__ t, const cplx* __restrict__ twb) {
    using PA = Plan2<LGA, false>;
    using PB = Plan2<LGB, true>;
    constexpr int LA = PA::L, LB = PB::L, S = LA + 1, SC = S * LB;
    if constexpr (PA::R2 * PB::R1 <= 16) {
        // lanes run over jb (rows, odd stride S: conflict-free), then over the a-blocks
        constexpr int NW = NCOMP * PA::R1 * PB::R2;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + threadIdx.x;
            if (NW % NT == 0 || w < NW) {
                const int jb = w % PB::R2, ba = (w / PB::R2) % PA::R1, c = w / (PB::R2 * PA::R1);
                block_smem<PA::R2, PB::R1, INV>(t + c * SC + jb * S + ba * PA::R2, 1, PB::R2 * S, twb, jb);
            }
        }
        __syncthreads();
    } else {
        // a stage 2 (contiguous sub-blocks of R2 points, no twiddles): lanes over rows
        auto a2 = [&]() {
            constexpr int NW = NCOMP * PA::R1 * LB;
#pragma unroll
            for (int w0 = 0; w0 < NW; w0 += NT) {
                const int w = w0 + threadIdx.x;
                if (NW % NT == 0 || w < NW) {
                    const int xb = w % LB, ba = (w / LB) % PA::R1, c = w / (LB * PA::R1);
                    stage_smem<PA::R2, INV, false>(t + c * SC + xb * S + ba * PA::R2, 1, nullptr, 0);
                }
            }
            __syncthreads();
        };
        // b stage 1 (sub-length LB, twiddles tw[k jb]): lanes over columns
        auto b1 = [&]() {
            constexpr int NW = NCOMP * LA * PB::R2;
#pragma unroll
            for (int w0 = 0; w0 < NW; w0 += NT) {
                const int w = w0 + threadIdx.x;
                if (NW % NT == 0 || w < NW) {
                    const int xa = w % LA, jb = (w / LA) % PB::R2, c = w / (LA * PB::R2);
                    stage_smem<PB::R1, INV, true>(t + c * SC + jb * S + xa, PB::R2 * S, twb, jb);
                }
            }
            __syncthreads();
        };
        if constexpr (INV) { b1(); a2(); } else { a2(); b1(); }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Forward FFT over axes 0,1 of the 4 component tiles t[c][x1][x0] (row stride L0+1), last stage written straight
// to field (component c at field + c*V, plane base xbase).  The tile must be complete (caller syncs before).
template <int LG0, int LG1, int NT>
__device__ __forceinline__ void plane_forward_store(cplx* __restrict__ tile, const cplx* __restrict__ tw0, const cplx* __restrict__ tw1,
                                                    cplx* __restrict__ field, long long V, long long xbase) {
    using PA = Plan2<LG0, false>;
    using PB = Plan2<LG1, true>;
    constexpr int L0 = PA::L, L1 = PB::L, S = L0 + 1, SC = S * L1;
    // a stage 1: points a = ja + m R2, twiddles tw0[k ja]; lanes over rows
    {
        constexpr int NW = 4 * PA::R2 * L1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + threadIdx.x;
            if (NW % NT == 0 || w < NW) {
                const int xb = w % L1, ja = (w / L1) % PA::R2, c = w / (L1 * PA::R2);
                stage_smem<PA::R1, false, true>(tile + c * SC + xb * S + ja, PA::R2, tw0, ja);
            }
        }
        __syncthreads();
    }
    plane_middle<LG0, LG1, 4, NT, false>(tile, tw1);
    // b stage 2 (no twiddles) -> global; lanes over x0: coalesced
    {
        constexpr int NW = 4 * L0 * PB::R1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + threadIdx.x;
            if (NW % NT == 0 || w < NW) {
                const int xa = w % L0, bb = (w / L0) % PB::R1, c = w / (L0 * PB::R1);
                const cplx* p = tile + c * SC + (bb * PB::R2) * S + xa;
                cplx v[PB::R2];
#pragma unroll
                for (int m = 0; m < PB::R2; m++) v[m] = p[m * S];
                bfly<PB::R2, false>(v);
                cplx* gq = field + (long long)c * V + xbase + ((bb * PB::R2) << LG0) + xa;
#pragma unroll
                for (int m = 0; m < PB::R2; m++) gq[m << LG0] = v[m];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Pass A: S1 (Delta, theta/F partials) + forward FFT over axes 0,1 of one (x2,x3) plane, all 4 components.
template <int LG0, int LG1, int NC, int NT>
__global__ void __launch_bounds__(NT, LGF_FA_MINB_DELTA) k_fa_delta_fwd(const cplx* __restrict__ links, cplx* __restrict__ field, double2* __restrict__ partials,
                                                     Geom G, FftTables T, const Ctl* __restrict__ ctl) {
    if (ctl->done) return;
    using PA = Plan2<LG0, false>;
    using PB = Plan2<LG1, true>;
    constexpr int L0 = PA::L, L1 = PB::L, S = L0 + 1, SC = S * L1, nP = L0 * L1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw0 = tile + 4 * SC;
    cplx* tw1 = tw0 + L0;
    __shared__ double red[64];
    const long long xbase = (long long)blockIdx.x << (LG0 + LG1);

    for (int i = threadIdx.x; i < L0; i += NT) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += NT) tw1[i] = T.tw[1][i];

    double th = 0, fs = 0;
#pragma unroll 1
    for (int e = threadIdx.x; e < nP; e += NT) {
        cplx f0, f1, f2, f3;
        double t_, f_;
        delta_site<NC>(links, G, xbase + e, f0, f1, f2, f3, t_, f_);
        th += t_; fs += f_;
        const int o = (e & (L0 - 1)) + (e >> LG0) * S;
        tile[o] = f0; tile[SC + o] = f1; tile[2 * SC + o] = f2; tile[3 * SC + o] = f3;
    }
    block_sum2(th, fs, red);     // contains a __syncthreads() after the tile writes
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(th, fs);
    __syncthreads();

    plane_forward_store<LG0, LG1, NT>(tile, tw0, tw1, field, G.V, xbase);
}

// Pass C: inverse FFT over axes 1,0 of one (x2,x3) plane for NCOMP components (blockIdx.x = plane * (4/NCOMP) + group).
// WRITE_G (NCOMP = 4): the last stage stays in the tile and the pass ends in S3, g(x) = GramSchmidt(1 + (alpha/2) X(x)),
// rows 0,1 written to gbuf (6 V-arrays) instead of X to field.
template <int LG0, int LG1, int NCOMP, int NT, bool WRITE_G>
__global__ void __launch_bounds__(NT, LGF_FA_MINB_INV) k_fa_inv(cplx* __restrict__ field, cplx* __restrict__ gbuf, double half_alpha, Geom G, FftTables T,
                                                                const Ctl* __restrict__ ctl) {
    static_assert(!WRITE_G || NCOMP == 4, "g needs all four components of X");
    if (ctl->done) return;
    using PA = Plan2<LG0, false>;
    using PB = Plan2<LG1, true>;
    constexpr int L0 = PA::L, L1 = PB::L, S = L0 + 1, SC = S * L1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw0 = tile + NCOMP * SC;
    cplx* tw1 = tw0 + L0;
    constexpr int NG = 4 / NCOMP;
    const long long xbase = (long long)(blockIdx.x / NG) << (LG0 + LG1);
    cplx* fbase = field + (long long)((blockIdx.x % NG) * NCOMP) * G.V + xbase;

    for (int i = threadIdx.x; i < L0; i += NT) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += NT) tw1[i] = T.tw[1][i];

    // global -> b stage 2 inverse (no twiddles) -> tile; lanes over x0
    {
        constexpr int NW = NCOMP * L0 * PB::R1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + threadIdx.x;
            if (NW % NT == 0 || w < NW) {
                const int xa = w % L0, bb = (w / L0) % PB::R1, c = w / (L0 * PB::R1);
                const cplx* gq = fbase + (long long)c * G.V + ((bb * PB::R2) << LG0) + xa;
                cplx v[PB::R2];
#pragma unroll
                for (int m = 0; m < PB::R2; m++) v[m] = gq[m << LG0];
                bfly<PB::R2, true>(v);
                cplx* p = tile + c * SC + (bb * PB::R2) * S + xa;
#pragma unroll
                for (int m = 0; m < PB::R2; m++) p[m * S] = v[m];
            }
        }
        __syncthreads();
    }
    plane_middle<LG0, LG1, NCOMP, NT, true>(tile, tw1);
    if constexpr (WRITE_G) {
        // a stage 1 inverse in place (lanes over rows: odd stride, conflict-free), then S3 per site
        constexpr int NW = NCOMP * PA::R2 * L1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + threadIdx.x;
            if (NW % NT == 0 || w < NW) {
                const int xb = w % L1, ja = (w / L1) % PA::R2, c = w / (L1 * PA::R2);
                stage_smem<PA::R1, true, true>(tile + c * SC + xb * S + ja, PA::R2, tw0, ja);
            }
        }
        __syncthreads();
        constexpr int nP = L0 * L1;
#pragma unroll 1
        for (int e = threadIdx.x; e < nP; e += NT) {
            const int o = (e & (L0 - 1)) + (e >> LG0) * S;
            cplx g[9];
            build_g(tile[o], tile[SC + o], tile[2 * SC + o], tile[3 * SC + o], half_alpha, g);
#pragma unroll
            for (int c = 0; c < 6; c++) gbuf[(long long)c * G.V + xbase + e] = g[c];
        }
        return;
    }
    // a stage 1 inverse (twiddles conj tw0[k ja]) -> global.  Lane order: each quarter-warp reads conflict-free and
    // each warp store covers whole 64 B (R2 = 4) or 128 B (R2 = 8) segments.
    {
        constexpr int NW = NCOMP * PA::R2 * L1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + threadIdx.x;
            if (NW % NT == 0 || w < NW) {
                int ja, xb;
                if constexpr (PA::R2 >= 8) { ja = w % PA::R2; xb = (w / PA::R2) % L1; }
                else { ja = (w / 8) % PA::R2; xb = (w % 8) + 8 * ((w / (8 * PA::R2)) % (L1 / 8)); }
                const int c = w / (PA::R2 * L1);
                const cplx* p = tile + c * SC + xb * S + ja;
                cplx v[PA::R1];
#pragma unroll
                for (int m = 0; m < PA::R1; m++) v[m] = p[m * PA::R2];
                stage_regs<PA::R1, true, true>(v, tw0, ja);
                cplx* gq = fbase + (long long)c * G.V + (xb << LG0) + ja;
#pragma unroll
                for (int m = 0; m < PA::R1; m++) gq[m * PA::R2] = v[m];
            }
        }
    }
}

// Pass B: forward over axes 2,3, filter, inverse over axes 3,2, for a chunk of C0 = 2^LGC consecutive x0 at fixed
// (component, x1).  tile[i3][i2][i0], S1 = C0, S2 = C0*L2 (+C0 when C0 < 8: keeps quarter-warps conflict-free).
template <int LG2, int LG3, int LGC, int NT>
__global__ void __launch_bounds__(NT, LGF_FA_MINB_MID) k_fa_mid(cplx* __restrict__ field, Geom G, FftTables T, double scale, const Ctl* __restrict__ ctl) {
    if (ctl->done) return;
    using PA = Plan2<LG2, false>;
    using PB = Plan2<LG3, true>;
    constexpr int L2 = PA::L, L3 = PB::L, C0 = 1 << LGC, S1 = C0, S2 = C0 * L2 + (C0 < 8 ? C0 : 0);
    static_assert(NT % C0 == 0, "a thread keeps its x0 offset");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw2 = tile + S2 * L3;
    cplx* tw3 = tw2 + L2;
    double* s2 = reinterpret_cast<double*>(tw3 + L3);
    double* s3 = s2 + L2;

    const int lgChunks = G.lg[0] - LGC;
    const int chunk = blockIdx.x & ((1 << lgChunks) - 1);
    const int x1 = (blockIdx.x >> lgChunks) & (G.L[1] - 1);
    const int comp = blockIdx.x >> (lgChunks + G.lg[1]);
    const int i0 = threadIdx.x % C0;
    cplx* gp = field + (long long)comp * G.V + (chunk << LGC) + ((long long)x1 << G.sh[1]) + i0;
    cplx* tl = tile + i0;
    const int sh2 = G.sh[2], sh3 = G.sh[3];

    for (int i = threadIdx.x; i < L2; i += NT) { tw2[i] = T.tw[2][i]; s2[i] = T.s[2][i]; }
    for (int i = threadIdx.x; i < L3; i += NT) { tw3[i] = T.tw[3][i]; s3[i] = T.s[3][i]; }
    const double s01 = T.s[0][(chunk << LGC) + i0] + T.s[1][x1];
    __syncthreads();

    // global -> axis-2 stage 1 (points i2 = ja + m R2, twiddles tw2[k ja]) -> tile
    {
        constexpr int NW = C0 * PA::R2 * L3;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + threadIdx.x;
            if (NW % NT == 0 || w < NW) {
                const int ja = (w / C0) % PA::R2, i3 = w / (C0 * PA::R2);
                const cplx* gq = gp + ((long long)ja << sh2) + ((long long)i3 << sh3);
                cplx v[PA::R1];
#pragma unroll
                for (int m = 0; m < PA::R1; m++) v[m] = gq[(long long)(m * PA::R2) << sh2];
                stage_regs<PA::R1, false, true>(v, tw2, ja);
                cplx* p = tl + ja * S1 + i3 * S2;
#pragma unroll
                for (int m = 0; m < PA::R1; m++) p[m * PA::R2 * S1] = v[m];
            }
        }
        __syncthreads();
    }
    // middle stages, forward and (after the filter) inverse
    auto middle = [&](auto inv_tag) {
        constexpr bool INV = decltype(inv_tag)::value;
        if constexpr (PA::R2 * PB::R1 <= 16) {
            constexpr int NW = C0 * PB::R2 * PA::R1;
#pragma unroll
            for (int w0 = 0; w0 < NW; w0 += NT) {
                const int w = w0 + threadIdx.x;
                if (NW % NT == 0 || w < NW) {
                    const int jb = (w / C0) % PB::R2, ba = w / (C0 * PB::R2);
                    block_smem<PA::R2, PB::R1, INV>(tl + ba * PA::R2 * S1 + jb * S2, S1, PB::R2 * S2, tw3, jb);
                }
            }
            __syncthreads();
        } else {
            auto a2 = [&]() {
                constexpr int NW = C0 * PA::R1 * L3;
#pragma unroll
                for (int w0 = 0; w0 < NW; w0 += NT) {
                    const int w = w0 + threadIdx.x;
                    if (NW % NT == 0 || w < NW) {
                        const int ba = (w / C0) % PA::R1, i3 = w / (C0 * PA::R1);
                        stage_smem<PA::R2, INV, false>(tl + ba * PA::R2 * S1 + i3 * S2, S1, nullptr, 0);
                    }
                }
                __syncthreads();
            };
            auto b1 = [&]() {
                constexpr int NW = C0 * L2 * PB::R2;
#pragma unroll
                for (int w0 = 0; w0 < NW; w0 += NT) {
                    const int w = w0 + threadIdx.x;
                    if (NW % NT == 0 || w < NW) {
                        const int i2 = (w / C0) % L2, jb = w / (C0 * L2);
                        stage_smem<PB::R1, INV, true>(tl + i2 * S1 + jb * S2, PB::R2 * S2, tw3, jb);
                    }
                }
                __syncthreads();
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
            const int w = w0 + threadIdx.x;
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
                    const double wgt = (p2 > 0.0) ? scale / p2 : 0.0;
                    v[m] = cscale(v[m], wgt);
                }
                bfly<PB::R2, true>(v);
#pragma unroll
                for (int m = 0; m < PB::R2; m++) p[m * S2] = v[m];
            }
        }
        __syncthreads();
    }
    middle(std::true_type{});
    // tile -> axis-2 stage 1 inverse -> global
    {
        constexpr int NW = C0 * PA::R2 * L3;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += NT) {
            const int w = w0 + threadIdx.x;
            if (NW % NT == 0 || w < NW) {
                const int ja = (w / C0) % PA::R2, i3 = w / (C0 * PA::R2);
                const cplx* p = tl + ja * S1 + i3 * S2;
                cplx v[PA::R1];
#pragma unroll
                for (int m = 0; m < PA::R1; m++) v[m] = p[m * PA::R2 * S1];
                stage_regs<PA::R1, true, true>(v, tw2, ja);
                cplx* gq = gp + ((long long)ja << sh2) + ((long long)i3 << sh3);
#pragma unroll
                for (int m = 0; m < PA::R1; m++) gq[(long long)(m * PA::R2) << sh2] = v[m];
            }
        }
    }
}

}  // namespace lgf
