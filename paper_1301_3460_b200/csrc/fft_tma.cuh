// fft_tma.cuh -- the FFT passes fed by the Tensor Memory Accelerator (cp.async.bulk.tensor + mbarrier), persistent, one CTA
// per SM:
//   k_tb_mid        pass B (axes 2,3: forward, p2max/p2 filter, inverse) for 16/32 extents: ring of three tiles, two thread
//                   groups, whole lines in registers
//   k_tm_mid        pass B for 64 x 64 tiles: the 128 KB tile in and out through the TMA unit, radix-16 stages
//   k_tr_mid        pass B for 32 x 64 / 64 x 32 tiles: ring of three 64 KB tiles, two thread groups, the same stages
//   k_ta_delta_fwd  pass A (S1 + forward FFT over axes 0,1) for 16/32-extent planes: the links staged 128 sites at a time
//
// Why: the plain-load passes of fft_fast.cuh are bound by latency, not by DRAM, the FP64 pipe or shared memory (ncu,
// profiles/r01_ncu_full_summary.txt: pass B DRAM 21 %, FP64 36 %, issue active 26 % at 7 warps per SM; pass A
// long_scoreboard 9.6 cycles per issue): a CTA loads its tile with dependent-latency global loads, transforms it, stores
// it, and nothing overlaps the three.  Here one elected thread issues a bulk tensor copy into a free shared-memory buffer
// and arms an mbarrier with the byte count; the copy costs neither registers nor issue slots and completes on the
// barrier while the warps work on other buffers.  Same arithmetic, same stored order, same results as the plain-load
// kernels (LGF_OPT_TMA = 0), against which every one of these is parity-tested.
#pragma once
#include <cuda.h>        // CUtensorMap (type only: the encoder is fetched through cudaGetDriverEntryPoint, lgf_api.cu)
#include <cstdint>
#include "fft_fast.cuh"

namespace lgf {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// makes the initialised barriers visible to the async proxy (the TMA unit) before the first copy is issued
__device__ __forceinline__ void mbar_init_fence() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LGF_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LGF_DONE_%=;\n"
        "bra LGF_WAIT_%=;\n"
        "LGF_DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 5-D tiled bulk tensor copy global -> shared, completion counted in bytes on the mbarrier
__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3, int c4) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* tm) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(tm) : "memory");
}

// Geometry of a pass-B tile in shared memory: dense [i3][i2][i0], exactly what the TMA box writes.
template <int LG2, int LG3, int LGC> struct TmaMidGeom {
    static constexpr int L2 = 1 << LG2, L3 = 1 << LG3, C0 = 1 << LGC;
    static constexpr int TILE = C0 * L2 * L3;                       // complex numbers per tile
    static constexpr unsigned TILE_BYTES = TILE * sizeof(cplx);
    static constexpr int NBUF = 3;
    // shared memory: three tile buffers, the p^2 tables of axes 2,3 (+ slack: the kernel rounds the dynamic
    // shared-memory base up to the 128 bytes a TMA destination needs)
    static constexpr size_t SMEM = (size_t)(NBUF * TILE) * sizeof(cplx) + (size_t)(L2 + L3) * 8 + 128;
};

#ifndef LGF_TB_NT
#define LGF_TB_NT 256
#endif

// The field as a 5-D tensor of reals for the TMA unit: (2 L0 reals, L1, L2, L3, 4 components); a pass-B tile is the box
// (2 C0, 1, L2, L3, 1) at (2 C0 chunk, x1, 0, 0, comp).  n_tiles = 4 L1 (L0 / C0); tile index = chunk + nChunks (x1 + L1 comp).
//
// One persistent CTA per SM, NT = 256 threads = two groups of 128 (a thread = one whole line in registers needs up to 255
// of them, so 8 warps is what an SM holds; with ONE group the FP64 dependency stalls are exposed: 60.6 us at 32^4, ncu
// "wait" 1.7 cycles per issue at 4 warps per SM).  The CTA's tiles form a sequence j = 0, 1, 2, ...; tile j is transformed
// by group j mod 2, in place, in buffer j mod 3.  When a group has finished tile j (phase 3 has read the buffer), its
// thread 0 starts the copy of tile j + 3 into the same buffer and arms that tile's mbarrier; the group that transforms
// tile j + 3 waits on it.  So each group always finds its next tile already in shared memory, the copies cost
// neither registers nor issue slots, and the two groups' phases interleave on the FP64 pipe.
// Barriers: tile j uses full[j mod 6] in phase j / 6 -- one barrier per (buffer, consuming group) pair, as 3 is odd and
// a buffer's consecutive tiles alternate between the groups.  Each barrier is therefore waited on by ONE group, phase after
// phase, and re-armed (tile j + 6) only after that group has consumed tile j: when the group arrives for phase k it has
// itself seen phase k - 1 complete, so a parity wait cannot be satisfied by an older phase.  (With one barrier per
// buffer the group that takes tile j + 3 had never waited for tile j, and its parity-1 wait would have passed on a
// barrier still in phase 0 had tile j not landed yet -- excluded only by timing.)  k_tr_mid uses the same scheme.
// Bank conflicts: the dense TMA layout makes lanes (i0, i3) and (i0, i3 + 1) of an axis-2 line collide (C0 = 4: 2-way) on
// the phase-1 reads only; phase 1 writes element m of line (i0, i3) at position m ^ (i3 & 1) -- inside the same line -- which
// makes its own writes, both accesses of phase 2 and the reads of phase 3 conflict-free.
template <int LG2, int LG3, int LGC, int NT>
__global__ void __launch_bounds__(NT, 1) k_tb_mid(const __grid_constant__ CUtensorMap tmap, cplx* __restrict__ field, Geom G, FftTables T,
                                                  double scale, Ctl* ctl, const double2* partials, FinArgs fa, int n_tiles) {
    static_assert(NT == 256, "two groups of 128 threads");
    pdl_enter();
    __shared__ int s_done;
    __shared__ __align__(8) uint64_t full[6];          // one per (buffer j mod 3, consuming group j mod 2): index j mod 6
    pass_b_entry<NT>(partials, fa, ctl, &s_done);
    using TG = TmaMidGeom<LG2, LG3, LGC>;
    constexpr int L2 = TG::L2, L3 = TG::L3, C0 = TG::C0, TILE = TG::TILE, GT = 128;
    constexpr int SW = (C0 < 8) ? 1 : 0;                 // C0 = 8: 128-byte rows, no conflicts, no swizzle
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // a TMA destination must be 128-byte aligned; the dynamic shared memory starts behind the static variables
    cplx* bufs = reinterpret_cast<cplx*>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));      // [3][TILE]
    double* s2 = reinterpret_cast<double*>(bufs + TG::NBUF * TILE);
    double* s3 = s2 + L2;
    for (int i = threadIdx.x; i < L2; i += NT) s2[i] = T.s[2][i];
    for (int i = threadIdx.x; i < L3; i += NT) s3[i] = T.s[3][i];
    const int lgChunks = G.lg[0] - LGC;
    const int n_seq = (n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;      // tiles of this CTA
    auto issue = [&](int j) {                            // one thread: arm the barrier of buffer j mod 3, start the copy of tile j
        const int tile = blockIdx.x + j * gridDim.x, b = j % 3;
        const int chunk = tile & ((1 << lgChunks) - 1);
        const int x1 = (tile >> lgChunks) & (G.L[1] - 1);
        const int comp = tile >> (lgChunks + G.lg[1]);
        mbar_expect_tx(&full[j % 6], TG::TILE_BYTES);
        tma_load_5d(bufs + b * TILE, &tmap, &full[j % 6], chunk << (LGC + 1), x1, 0, 0, comp);
    };
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < 6; i++) mbar_init(&full[i], 1);
        mbar_init_fence();
        // a copy in flight must never outlive its CTA: nothing is issued when the run is already over
        if (!s_done)
            for (int j = 0; j < 3 && j < n_seq; j++) issue(j);
    }
    __syncthreads();
    if (s_done) return;                                  // one reading per CTA, behind a barrier (pass_b_entry)
    const int sh2 = G.sh[2], sh3 = G.sh[3];
    const Grp g{(int)threadIdx.x % GT, 1 + (int)threadIdx.x / GT};      // named barriers 1 and 2
#pragma unroll 1
    for (int j = threadIdx.x / GT; j < n_seq; j += 2) {
        const int tile = blockIdx.x + j * gridDim.x, b = j % 3;
        const int chunk = tile & ((1 << lgChunks) - 1);
        const int x1 = (tile >> lgChunks) & (G.L[1] - 1);
        const int comp = tile >> (lgChunks + G.lg[1]);
        cplx* gbase = field + (long long)comp * G.V + (chunk << LGC) + ((long long)x1 << G.sh[1]);
        cplx* tl = bufs + b * TILE;
        mbar_wait(&full[j % 6], (j / 6) & 1);
        // phase 1: lines along axis 2, one per (i0, i3): forward, in place (element m -> position m ^ (i3 & 1))
#pragma unroll 1
        for (int ln = g.tid; ln < C0 * L3; ln += GT) {
            const int i0 = ln % C0, i3 = ln / C0;
            cplx* q = tl + i0 + i3 * (C0 * L2);
            cplx v[L2];
#pragma unroll
            for (int m = 0; m < L2; m++) v[m] = q[m * C0];
            line_fft<LG2, false, false>(v);
            const int par = SW * (i3 & 1) * C0;
            cplx* qe = q + par;                          // even m: position m + par
            cplx* qo = q - par;                          // odd m:  position m - par
#pragma unroll
            for (int m = 0; m < L2; m++) ((m & 1) ? qo : qe)[m * C0] = v[m];
        }
        gsync<GT>(g);
        // phase 2: lines along axis 3, one per (i0, i2): forward, filter X~ = (p2max / (V p2)) Delta~ at the stored
        // positions (zero mode -> 0), inverse                                                       [north_star step 2]
#pragma unroll 1
        for (int ln = g.tid; ln < C0 * L2; ln += GT) {
            const int i0 = ln % C0, i2 = ln / C0;
            // element (i2, i3 = m) sits at position i2 ^ (m & 1) of its axis-2 line
            cplx* pe = tl + i0 + i2 * C0;
            cplx* po = tl + i0 + (i2 ^ SW) * C0;
            cplx v[L3];
#pragma unroll
            for (int m = 0; m < L3; m++) v[m] = ((m & 1) ? po : pe)[m * (C0 * L2)];
            line_fft<LG3, true, false>(v);
            const double s012 = T.s[0][(chunk << LGC) + i0] + T.s[1][x1] + s2[i2];
#pragma unroll
            for (int m = 0; m < L3; m++) {
                const double p2 = s012 + s3[m];
                v[m] = cscale(v[m], (real)filter_weight(scale, p2));
            }
            line_fft<LG3, true, true>(v);
#pragma unroll
            for (int m = 0; m < L3; m++) ((m & 1) ? po : pe)[m * (C0 * L2)] = v[m];
        }
        gsync<GT>(g);
        // phase 3: lines along axis 2 again: inverse, straight to global memory
#pragma unroll 1
        for (int ln = g.tid; ln < C0 * L3; ln += GT) {
            const int i0 = ln % C0, i3 = ln / C0;
            const cplx* q = tl + i0 + i3 * (C0 * L2);
            const int par = SW * (i3 & 1) * C0;
            const cplx* qe = q + par;
            const cplx* qo = q - par;
            cplx v[L2];
#pragma unroll
            for (int m = 0; m < L2; m++) v[m] = ((m & 1) ? qo : qe)[m * C0];
            line_fft<LG2, false, true>(v);
            cplx* gq = gbase + i0 + ((long long)i3 << sh3);
#pragma unroll
            for (int m = 0; m < L2; m++) st_field(gq + ((long long)m << sh2), v[m]);
        }
        gsync<GT>(g);                                    // every thread of the group has read the buffer
        if (g.tid == 0 && j + 3 < n_seq) issue(j + 3);   // same buffer, next tile of the chain
    }
}


// ---------------------------------------------------------------------------------------------------------------
// Pass B for (x2,x3) tiles with a 64 extent: the tile (2^LGC x0 sites x L2 x L3, 128 KB) fills the SM, so there is one
// buffer and no second tile in flight -- but the plain-load version of this pass (k_fa_mid) is bound by the L1 queue for
// global memory instructions (ncu at 64^4: lg_throttle 4.1 cycles per issue; a warp-wide load of 2-site chunks touches 16
// different 128-byte lines).  Here the tile comes in and goes out through the TMA unit (one 5-D bulk tensor copy each
// way), which takes the 32/64-byte rows off the LSU, and the stages are those of k_fa_mid with PlanM's radices
// (16 x 4 | 4 x 16 at 64: the tile crosses shared memory 8 times).  The TMA box is dense, [i3][i2][i0]; between the
// first and the last stage element (i2, i3) of an (x2,x3) plane sits at position i2 ^ (i3 & SWM), SWM = 8/C0 - 1, inside
// its own axis-2 line, which makes every stage's accesses conflict-free without padding.
__device__ __forceinline__ void tma_store_5d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2, int c3, int c4) {
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5, %6}], [%1];"
                 ::"l"(tm), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int LG2, int LG3, int LGC> struct TmaBigGeom {
    static constexpr int L2 = 1 << LG2, L3 = 1 << LG3, C0 = 1 << LGC;
    static constexpr int TILE = C0 * L2 * L3;
    static constexpr unsigned TILE_BYTES = TILE * sizeof(cplx);
    static constexpr size_t SMEM = (size_t)(TILE + L2 + L3) * sizeof(cplx) + (size_t)(L2 + L3) * 8 + 128;
};

// The stages of pass B on one dense tile (entry: the TMA box [i3][i2][i0]; exit: the same layout, transformed), run by
// the GT threads of group g; tl = tile + the thread's x0 offset (g.tid % C0).  Ends behind the group's last writes (the
// caller fences and synchronises before the tile is handed to the TMA unit).
template <int LG2, int LG3, int LGC, int GT, int BAR>
__device__ __forceinline__ void mid_tile_stages(cplx* tl, const cplx* tw2, const cplx* tw3, const double* s2, const double* s3, double s01, double scale,
                                                int gtid) {
    using PA = PlanM<LG2, false>;
    using PB = PlanM<LG3, true>;
    constexpr int L2 = 1 << LG2, L3 = 1 << LG3, C0 = 1 << LGC;
    constexpr int SI2 = C0, SI3 = C0 * L2;               // element strides of i2 and i3 in the dense tile
    constexpr int SWM = (C0 < 8) ? (8 / C0 - 1) : 0;
    static_assert(PA::R2 == 4 && PB::R1 == 4, "one 16-point block between the axes");
    static_assert(GT % C0 == 0, "a thread keeps its x0 offset");
    // axis-2 stage 1 (points i2 = ja + m R2, twiddles tw2[k ja]): dense in, swizzled out
    {
        constexpr int NW = C0 * PA::R2 * L3, NI = (NW + GT - 1) / GT;
        static_assert(NW % GT == 0, "whole items per thread");
        cplx v[NI][PA::R1];
#pragma unroll
        for (int k = 0; k < NI; k++) {
            const int w = k * GT + gtid;
            const int ja = (w / C0) % PA::R2, i3 = w / (C0 * PA::R2);
            const cplx* p = tl + ja * SI2 + i3 * SI3;
#pragma unroll
            for (int m = 0; m < PA::R1; m++) v[k][m] = p[m * PA::R2 * SI2];
            stage_regs<PA::R1, false, true>(v[k], tw2, ja);
        }
        gsync_c<GT, BAR>();
#pragma unroll
        for (int k = 0; k < NI; k++) {
            const int w = k * GT + gtid;
            const int ja = (w / C0) % PA::R2, i3 = w / (C0 * PA::R2);
            // position (ja + 4 m) ^ sw = (ja ^ (sw & 3)) + 4 (m ^ (sw >> 2)): two base pointers, static offsets
            const int sw = i3 & SWM, hb = (sw >> 2) * 4 * SI2;
            cplx* pe = tl + (ja ^ (sw & 3)) * SI2 + i3 * SI3 + hb;
            cplx* po = pe - 2 * hb;
#pragma unroll
            for (int m = 0; m < PA::R1; m++) ((m & 1) ? po : pe)[m * PA::R2 * SI2] = v[k][m];
        }
        gsync_c<GT, BAR>();
    }
    // 16-point block: last stage of axis 2 (contiguous sub-blocks of 4) x first stage of axis 3 (points jb + mb R2b)
    auto block = [&](auto inv_tag) {
        constexpr bool INV = decltype(inv_tag)::value;
        constexpr int NW = C0 * PB::R2 * PA::R1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += GT) {
            const int w = w0 + gtid;
            if (NW % GT == 0 || w < NW) {
                const int jb = (w / C0) % PB::R2, ba = w / (C0 * PB::R2);
                const int sw = jb & SWM;
                cplx v[4][4];                        // [mb][ma]
#pragma unroll
                for (int mb = 0; mb < 4; mb++)
#pragma unroll
                    for (int ma = 0; ma < 4; ma++) v[mb][ma] = tl[((ba * 4 + ma) ^ sw) * SI2 + (jb + mb * PB::R2) * SI3];
                if constexpr (!INV) {
#pragma unroll
                    for (int mb = 0; mb < 4; mb++) bfly<4, false>(v[mb]);
                }
#pragma unroll
                for (int ma = 0; ma < 4; ma++) {
                    cplx c[4];
#pragma unroll
                    for (int mb = 0; mb < 4; mb++) c[mb] = v[mb][ma];
                    stage_regs<4, INV, true>(c, tw3, jb);
#pragma unroll
                    for (int mb = 0; mb < 4; mb++) v[mb][ma] = c[mb];
                }
                if constexpr (INV) {
#pragma unroll
                    for (int mb = 0; mb < 4; mb++) bfly<4, true>(v[mb]);
                }
#pragma unroll
                for (int mb = 0; mb < 4; mb++)
#pragma unroll
                    for (int ma = 0; ma < 4; ma++) tl[((ba * 4 + ma) ^ sw) * SI2 + (jb + mb * PB::R2) * SI3] = v[mb][ma];
            }
        }
        gsync_c<GT, BAR>();
    };
    block(std::false_type{});
    // axis-3 stage 2 forward, S2b filter X~ = (p2max / (V p2)) Delta~ at the stored positions (zero mode -> 0), axis-3
    // stage 2 inverse, on the same registers                                                   [north_star step 2]
    {
        constexpr int NW = C0 * L2 * PB::R1;
#pragma unroll
        for (int w0 = 0; w0 < NW; w0 += GT) {
            const int w = w0 + gtid;
            if (NW % GT == 0 || w < NW) {
                const int i2 = (w / C0) % L2, bb = w / (C0 * L2);
                cplx v[PB::R2];
#pragma unroll
                for (int m = 0; m < PB::R2; m++) v[m] = tl[(i2 ^ (m & SWM)) * SI2 + (bb * PB::R2 + m) * SI3];
                bfly<PB::R2, false>(v);
                const double s012 = s01 + s2[i2];
#pragma unroll
                for (int m = 0; m < PB::R2; m++) {
                    const double p2 = s012 + s3[bb * PB::R2 + m];
                    v[m] = cscale(v[m], (real)filter_weight(scale, p2));
                }
                bfly<PB::R2, true>(v);
#pragma unroll
                for (int m = 0; m < PB::R2; m++) tl[(i2 ^ (m & SWM)) * SI2 + (bb * PB::R2 + m) * SI3] = v[m];
            }
        }
        gsync_c<GT, BAR>();
    }
    block(std::true_type{});
    // axis-2 stage 1 inverse: swizzled in, dense out, then the tile goes back through the TMA unit
    {
        constexpr int NW = C0 * PA::R2 * L3, NI = (NW + GT - 1) / GT;
        cplx v[NI][PA::R1];
#pragma unroll
        for (int k = 0; k < NI; k++) {
            const int w = k * GT + gtid;
            const int ja = (w / C0) % PA::R2, i3 = w / (C0 * PA::R2);
            const int sw = i3 & SWM, hb = (sw >> 2) * 4 * SI2;
            const cplx* pe = tl + (ja ^ (sw & 3)) * SI2 + i3 * SI3 + hb;
            const cplx* po = pe - 2 * hb;
#pragma unroll
            for (int m = 0; m < PA::R1; m++) v[k][m] = ((m & 1) ? po : pe)[m * PA::R2 * SI2];
            stage_regs<PA::R1, true, true>(v[k], tw2, ja);
        }
        gsync_c<GT, BAR>();
#pragma unroll
        for (int k = 0; k < NI; k++) {
            const int w = k * GT + gtid;
            const int ja = (w / C0) % PA::R2, i3 = w / (C0 * PA::R2);
            cplx* p = tl + ja * SI2 + i3 * SI3;
#pragma unroll
            for (int m = 0; m < PA::R1; m++) p[m * PA::R2 * SI2] = v[k][m];
        }
    }
}

template <int LG2, int LG3, int LGC, int NT>
__global__ void __launch_bounds__(NT, 1) k_tm_mid(const __grid_constant__ CUtensorMap tmap, cplx* __restrict__ field, Geom G, FftTables T,
                                                  double scale, Ctl* ctl, const double2* partials, FinArgs fa, int n_tiles) {
    pdl_enter();
    __shared__ int s_done;
    __shared__ __align__(8) uint64_t full;
    pass_b_entry<NT>(partials, fa, ctl, &s_done);
    using PA = PlanM<LG2, false>;
    using PB = PlanM<LG3, true>;
    using TG = TmaBigGeom<LG2, LG3, LGC>;
    constexpr int L2 = TG::L2, L3 = TG::L3, C0 = TG::C0, TILE = TG::TILE;
    constexpr int SI2 = C0, SI3 = C0 * L2;               // element strides of i2 and i3 in the dense tile
    constexpr int SWM = (C0 < 8) ? (8 / C0 - 1) : 0;
    static_assert(PA::R2 == 4 && PB::R1 == 4, "one 16-point block between the axes");
    static_assert(NT % C0 == 0, "a thread keeps its x0 offset");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tile = reinterpret_cast<cplx*>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));
    cplx* tw2 = tile + TILE;
    cplx* tw3 = tw2 + L2;
    double* s2 = reinterpret_cast<double*>(tw3 + L3);
    double* s3 = s2 + L2;
    for (int i = threadIdx.x; i < L2; i += NT) { tw2[i] = T.tw[2][i]; s2[i] = T.s[2][i]; }
    for (int i = threadIdx.x; i < L3; i += NT) { tw3[i] = T.tw[3][i]; s3[i] = T.s[3][i]; }
    const int lgChunks = G.lg[0] - LGC;
    if (threadIdx.x == 0) { mbar_init(&full, 1); mbar_init_fence(); }
    __syncthreads();
    if (s_done) return;                                  // one reading per CTA, behind a barrier (pass_b_entry)
    const int i0 = threadIdx.x % C0;
    cplx* tl = tile + i0;
    int it = 0;
#pragma unroll 1
    for (int tileno = blockIdx.x; tileno < n_tiles; tileno += gridDim.x, it++) {
        const int chunk = tileno & ((1 << lgChunks) - 1);
        const int x1 = (tileno >> lgChunks) & (G.L[1] - 1);
        const int comp = tileno >> (lgChunks + G.lg[1]);
        if (threadIdx.x == 0) {
            mbar_expect_tx(&full, TG::TILE_BYTES);
            tma_load_5d(tile, &tmap, &full, chunk << (LGC + 1), x1, 0, 0, comp);
        }
        const double s01 = T.s[0][(chunk << LGC) + i0] + T.s[1][x1];
        mbar_wait(&full, it & 1);
        mid_tile_stages<LG2, LG3, LGC, NT, 0>(tl, tw2, tw3, s2, s3, s01, scale, (int)threadIdx.x);
        fence_proxy_async();                             // the generic-proxy writes above, before the async proxy reads them
        __syncthreads();
        if (threadIdx.x == 0) {
            tma_store_5d(&tmap, tile, chunk << (LGC + 1), x1, 0, 0, comp);
            tma_store_wait_read();                       // the buffer is free again once the store has read it
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) tma_store_wait_all();
}

}  // namespace lgf

namespace lgf {

// ---------------------------------------------------------------------------------------------------------------
// Pass B for 32 x 64 and 64 x 32 tiles as a RING: tiles of HALF the x0 chunk of k_tm_mid (64 KB: two sites x 32 x 64),
// three buffers, NT = 512 threads = two groups of 256.  (Measured: 74.6 against 106.3 us at 32^3 x 64.  For 64 x 64 the
// half chunk is ONE site, the rows of the TMA box are 16 bytes, and the ring measured slower than k_tm_mid -- 1065
// against 999 us at 64^4 -- so that shape keeps the single-buffered kernel.)  As in k_tb_mid, tile j of the CTA's sequence is
// transformed in place in buffer j mod 3 by group j mod 2 (the stages of mid_tile_stages on the group's named barrier),
// goes back to the field by a bulk tensor store, and when that store has read the buffer the group's thread 0 starts the
// copy of tile j + 3 into it.  So the load and the store of a tile overlap the other group's stages instead of standing
// in front of and behind the tile's own (k_tm_mid: about a quarter of the tile's time).  The CTA takes its tiles in
// PAIRS of neighbouring x0 chunks (j and j + 1 share their 32- or 64-byte sectors), so the second copy of a pair finds its
// sectors in L2 and the two partial-sector stores meet there before they go to DRAM.
template <int LG2, int LG3, int LGC> struct TmaRingGeom {
    static constexpr int L2 = 1 << LG2, L3 = 1 << LG3, C0 = 1 << LGC;
    static constexpr int TILE = C0 * L2 * L3;
    static constexpr unsigned TILE_BYTES = TILE * sizeof(cplx);
    static constexpr size_t SMEM = (size_t)(3 * TILE + L2 + L3) * sizeof(cplx) + (size_t)(L2 + L3) * 8 + 128;
};

template <int LG2, int LG3, int LGC, int NT>
__global__ void __launch_bounds__(NT, 1) k_tr_mid(const __grid_constant__ CUtensorMap tmap, cplx* __restrict__ field, Geom G, FftTables T,
                                                  double scale, Ctl* ctl, const double2* partials, FinArgs fa, int n_tiles) {
    static_assert(NT == 512, "two groups of 256 threads");
    pdl_enter();
    __shared__ int s_done;
    __shared__ __align__(8) uint64_t full[6];          // one per (buffer j mod 3, consuming group j mod 2): index j mod 6
    pass_b_entry<NT>(partials, fa, ctl, &s_done);
    using TG = TmaRingGeom<LG2, LG3, LGC>;
    constexpr int L2 = TG::L2, L3 = TG::L3, C0 = TG::C0, TILE = TG::TILE, GT = 256;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* bufs = reinterpret_cast<cplx*>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));      // [3][TILE]
    cplx* tw2 = bufs + 3 * TILE;
    cplx* tw3 = tw2 + L2;
    double* s2 = reinterpret_cast<double*>(tw3 + L3);
    double* s3 = s2 + L2;
    for (int i = threadIdx.x; i < L2; i += NT) { tw2[i] = T.tw[2][i]; s2[i] = T.s[2][i]; }
    for (int i = threadIdx.x; i < L3; i += NT) { tw3[i] = T.tw[3][i]; s3[i] = T.s[3][i]; }
    const int lgChunks = G.lg[0] - LGC;
    // tile j of this CTA: the (j & 1)-th of the pair blockIdx.x + (j >> 1) gridDim.x
    const int n_pairs = n_tiles >> 1;
    const int n_seq = 2 * ((n_pairs - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x);
    auto tile_of = [&](int j) { return 2 * ((int)blockIdx.x + (j >> 1) * (int)gridDim.x) + (j & 1); };
    auto issue = [&](int j) {
        const int tile = tile_of(j), b = j % 3;
        const int chunk = tile & ((1 << lgChunks) - 1);
        const int x1 = (tile >> lgChunks) & (G.L[1] - 1);
        const int comp = tile >> (lgChunks + G.lg[1]);
        mbar_expect_tx(&full[j % 6], TG::TILE_BYTES);
        tma_load_5d(bufs + b * TILE, &tmap, &full[j % 6], chunk << (LGC + 1), x1, 0, 0, comp);
    };
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < 6; i++) mbar_init(&full[i], 1);
        mbar_init_fence();
        if (!s_done)
            for (int j = 0; j < 3 && j < n_seq; j++) issue(j);
    }
    __syncthreads();
    if (s_done) return;                                  // one reading per CTA, behind a barrier (pass_b_entry)
    const int grp = threadIdx.x / GT, gtid = threadIdx.x % GT;
    const int i0 = gtid % C0;
#pragma unroll 1
    for (int j = grp; j < n_seq; j += 2) {
        const int tile = tile_of(j), b = j % 3;
        const int chunk = tile & ((1 << lgChunks) - 1);
        const int x1 = (tile >> lgChunks) & (G.L[1] - 1);
        const int comp = tile >> (lgChunks + G.lg[1]);
        cplx* tbuf = bufs + b * TILE;
        const double s01 = T.s[0][(chunk << LGC) + i0] + T.s[1][x1];
        mbar_wait(&full[j % 6], (j / 6) & 1);
        if (grp == 0) mid_tile_stages<LG2, LG3, LGC, GT, 1>(tbuf + i0, tw2, tw3, s2, s3, s01, scale, gtid);
        else mid_tile_stages<LG2, LG3, LGC, GT, 2>(tbuf + i0, tw2, tw3, s2, s3, s01, scale, gtid);
        fence_proxy_async();                             // the generic-proxy writes above, before the async proxy reads them
        if (grp == 0) gsync_c<GT, 1>(); else gsync_c<GT, 2>();
        if (gtid == 0) {
            tma_store_5d(&tmap, tbuf, chunk << (LGC + 1), x1, 0, 0, comp);
            tma_store_wait_read();                       // this group's only outstanding store has read the buffer ...
            if (j + 3 < n_seq) issue(j + 3);             // ... which takes the next tile of its chain
        }
    }
    if (gtid == 0) tma_store_wait_all();
}

// ---------------------------------------------------------------------------------------------------------------
// Pass A (S1 + forward FFT over axes 0,1) with the links staged by the TMA unit.
//
// k_fa_delta_fwd is bound by the latency of S1's loads (ncu, profiles/r01: long_scoreboard 9.6 cycles per issue at 14.5
// warps per SM; 48 loads per site, each warp waits for all of them before it computes).  Here one persistent CTA per SM
// walks over its (x2,x3) planes and the links arrive by bulk tensor copies, stage by stage, while the warps work: a
// stage is 128 consecutive sites of the plane (R = 128/L0 rows) and holds, as dense arrays [stream][site],
//   own   the 4 NC streams of the sites' own links U_mu(x)                       one copy, box (256 reals, 1 plane, 4 NC streams)
//   nb2   U_2(x-2): the NC streams of direction 2 in the plane (x2-1, x3)        box (256, 1, NC)
//   nb3   U_3(x-3): direction 3 in the plane (x2, x3-1)                          box (256, 1, NC)
//   row1  U_1 of the row below the stage's first row (U_1(x-1) of that row)      box (2 L0, 1, NC)
// (U_0(x-0), and U_1(x-1) of the other rows, are inside `own`).  The links are a 3-D tensor for the TMA unit:
// (2 L0 L1 reals of a plane, L2 L3 planes, 4 NC streams).  NT = 256 threads = two groups of 128, a thread = one site of
// a stage; group g takes the stages s = g (mod 2) into ITS OWN buffer, and when all its threads have read the buffer its
// thread 0 starts the copies of stage s + 2 -- of the same plane or the CTA's next one -- and arms the buffer's mbarrier.
// So two stages (150 KB at 32 x 32, fp64) are always in flight or being consumed, also while all warps transform the
// finished tile, and no warp ever waits on a global load.
// The planes are walked from the LAST one down: the link update before this kernel walks the lattice upwards, so the
// last ~100 MB of links it wrote are still in L2 and this kernel starts on exactly those (measured at 32^4: 92.9 against
// 97.3 us; walking the update downwards instead gives pass A the same hits but costs the update its own on X).
struct LinkMaps { CUtensorMap own, nb, row; };

// Sites per stage: 128 -- a thread = one site, each group owns one buffer.  A variant with 64-site stages (two threads per
// site, summed by a lane-pair shuffle, two buffers per group so that a group's next stage lands while it works on the
// current one) was built, measured and removed in round 3 (history: commit d75b9c7): at 32^4 98.6-99.4 against
// 100.6-101.7 us.  The finer pipeline does not pay, because what is exposed is not the per-buffer load/compute
// cycle but the transform of the finished tile: leaving phases out gives 78.5 us for the staged copies alone (0.92 of the
// measured HBM peak on the kernel's 470 MB), 90.6 with the transform, 100 with S1 as well -- while all warps transform a
// tile the 150 KB of stage buffers fill up and the SM's share of HBM idles for the rest of the phase; a second tile or
// deeper buffers do not fit (222 KB used), and pulling stages further ahead into L2 with cp.async.bulk.prefetch.tensor
// made it slower at every distance tried (102.5 at one stage ahead of the window, 119 at a plane ahead).
constexpr int TA_SS = 128;
template <int LG0, int LG1, int NC> struct TmaPlaneGeom {
    static constexpr int L0 = 1 << LG0, L1 = 1 << LG1, S = L0 + 1, SC = S * L1, nP = L0 * L1;
    static constexpr int SS = TA_SS;                                 // sites per stage = threads per group
    static constexpr int NST = nP / SS;                              // stages per plane
    static constexpr int OWN = 4 * NC * SS, NB = NC * SS, ROW = NC * L0;      // complex numbers
    static constexpr int STAGE = OWN + 2 * NB + ROW;
    static constexpr unsigned STAGE_BYTES = STAGE * sizeof(cplx);
    static_assert(SS % L0 == 0, "a stage is whole x0 rows");
    static_assert(NST >= 2 && NST % 2 == 0, "each group takes every other stage");
    static_assert((OWN * sizeof(cplx)) % 128 == 0 && (NB * sizeof(cplx)) % 128 == 0 && (STAGE * sizeof(cplx)) % 128 == 0, "TMA destinations are 128-byte aligned");
    static constexpr size_t SMEM = (size_t)(2 * STAGE + 4 * SC + L0 + L1) * sizeof(cplx) + 128;
};

__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

template <int NC> __device__ __forceinline__ void load_link_smem(const cplx* __restrict__ p, int stride, cplx (&u)[9]) {
#pragma unroll
    for (int c = 0; c < NC; c++) u[c] = p[c * stride];
    if (NC == 6) third_row(u);
}

template <int LG0, int LG1, int NC, int NT>
__global__ void __launch_bounds__(NT, 1) k_ta_delta_fwd(const __grid_constant__ LinkMaps maps, cplx* __restrict__ field, double2* __restrict__ partials,
                                                        Geom G, FftTables T, const Ctl* __restrict__ ctl, int n_planes) {
    static_assert(NT == 256, "two groups of 128 threads");
    pdl_enter();
    if (ctl->done) return;                               // uniform over the grid; nothing has been issued yet
    using PG = TmaPlaneGeom<LG0, LG1, NC>;
    constexpr int L0 = PG::L0, L1 = PG::L1, S = PG::S, SC = PG::SC, SS = PG::SS, NST = PG::NST, GT = 128;
    static_assert(SS == GT, "a thread of a group = one site of its stage");
    __shared__ __align__(8) uint64_t full[2];            // one per group: only that group waits on it, phase after phase
    __shared__ double red[64];
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* stage = reinterpret_cast<cplx*>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));      // [2][STAGE]
    cplx* tile = stage + 2 * PG::STAGE;
    cplx* tw0 = tile + 4 * SC;
    cplx* tw1 = tw0 + L0;
    for (int i = threadIdx.x; i < L0; i += NT) tw0[i] = T.tw[0][i];
    for (int i = threadIdx.x; i < L1; i += NT) tw1[i] = T.tw[1][i];
    const int n_seq = (n_planes - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;      // planes of this CTA
    const int n_stage = n_seq * NST;
    // Stage t of this CTA: plane blockIdx.x + (t / NST) gridDim.x, sites [(t % NST) SS, ...).  Group g = t & 1 takes it as
    // its k-th stage, k = t >> 1, in its own buffer.
    auto issue = [&](int t) {
        const int plane = n_planes - 1 - ((int)blockIdx.x + (t / NST) * (int)gridDim.x), s = t % NST, b = t & 1;
        const int x2 = plane & (G.L[2] - 1), x3 = plane >> G.lg[2];
        const int pl2 = ((x2 + G.L[2] - 1) & (G.L[2] - 1)) + (x3 << G.lg[2]);
        const int pl3 = x2 + (((x3 + G.L[3] - 1) & (G.L[3] - 1)) << G.lg[2]);
        const int r0 = 2 * SS * s;                                      // first real of the stage inside the plane
        const int rowb = 2 * L0 * (((s * (SS / L0)) + L1 - 1) & (L1 - 1));   // the row below the stage's first row
        cplx* d = stage + b * PG::STAGE;
        mbar_expect_tx(&full[b], PG::STAGE_BYTES);
        tma_load_3d(d, &maps.own, &full[b], r0, plane, 0);
        tma_load_3d(d + PG::OWN, &maps.nb, &full[b], r0, pl2, 2 * NC);
        tma_load_3d(d + PG::OWN + PG::NB, &maps.nb, &full[b], r0, pl3, 3 * NC);
        tma_load_3d(d + PG::OWN + 2 * PG::NB, &maps.row, &full[b], rowb, plane, NC);
    };
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1); mbar_init(&full[1], 1);
        mbar_init_fence();
        for (int t = 0; t < 2 && t < n_stage; t++) issue(t);
    }
    __syncthreads();
    const int grp = threadIdx.x / GT;
    const Grp g{(int)threadIdx.x % GT, 1 + grp};
    const Grp all{(int)threadIdx.x, 0};
    const int j = g.tid;                                               // a thread's site of the stage
    const int jx = j & (L0 - 1), jr = j >> LG0;                        // x0, row inside the stage
    const int jm0 = (j & ~(L0 - 1)) | ((jx + L0 - 1) & (L0 - 1));      // x - 0 (periodic inside the row)
#pragma unroll 1
    for (int q = 0; q < n_seq; q++) {
        const int plane = n_planes - 1 - ((int)blockIdx.x + q * (int)gridDim.x);
        double th = 0, fs = 0;
#pragma unroll 1
        for (int s = grp; s < NST; s += 2) {
            const int t = q * NST + s, k = t >> 1, b = grp;
            const cplx* own = stage + b * PG::STAGE;
            const cplx* nb2 = own + PG::OWN;
            const cplx* nb3 = nb2 + PG::NB;
            const cplx* row1 = nb3 + PG::NB;
            mbar_wait(&full[b], k & 1);
            cplx d01 = mk(0, 0), d02 = mk(0, 0), d12 = mk(0, 0);
            real i0 = 0, i1 = 0, i2 = 0, retr = 0;
            cplx u[9];
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {                           // the site's own links: - U_mu(x)
                load_link_smem<NC>(own + mu * NC * SS + j, SS, u);
                retr += u[0].x + u[4].x + u[8].x;
                acc_link(u, real(-1), d01, d02, d12, i0, i1, i2);
            }
            load_link_smem<NC>(own + jm0, SS, u);                      // the backward neighbours: + U_mu(x-mu)
            acc_link(u, real(1), d01, d02, d12, i0, i1, i2);
            load_link_smem<NC>(jr == 0 ? row1 + jx : own + NC * SS + j - L0, jr == 0 ? L0 : SS, u);
            acc_link(u, real(1), d01, d02, d12, i0, i1, i2);
            load_link_smem<NC>(nb2 + j, SS, u);
            acc_link(u, real(1), d01, d02, d12, i0, i1, i2);
            load_link_smem<NC>(nb3 + j, SS, u);
            acc_link(u, real(1), d01, d02, d12, i0, i1, i2);
            const real tr3 = real(2.0 / 3.0) * (i0 + i1 + i2);
            const real e0 = real(2) * i0 - tr3, e1 = real(2) * i1 - tr3, e2 = real(2) * i2 - tr3;
            const int o = jx + (s * (SS / L0) + jr) * S;
            th += (double)(real(2) * (cnorm2(d01) + cnorm2(d02) + cnorm2(d12)) + e0 * e0 + e1 * e1 + e2 * e2);
            fs += (double)retr;
            tile[o] = d01; tile[SC + o] = d02; tile[2 * SC + o] = d12; tile[3 * SC + o] = mk(e0, e1);
            gsync<GT>(g);                                              // every thread of the group has read the buffer
            if (g.tid == 0 && t + 2 < n_stage) issue(t + 2);
        }
        group_sum2<NT>(th, fs, red, all);                              // its barrier also completes the tile
        if (threadIdx.x == 0) partials[plane] = make_double2(th, fs);
        gsync<NT>(all);
        plane_forward_store<LG0, LG1, NT>(tile, tw0, tw1, field, G.V, (long long)plane << (LG0 + LG1), all);
        gsync<NT>(all);                                                // the tile is rewritten by the next plane's S1
    }
}

}  // namespace lgf
