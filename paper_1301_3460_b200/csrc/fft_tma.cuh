// fft_tma.cuh -- pass B (axes 2,3: forward, p2max/p2 filter, inverse) on tiles staged by the Tensor Memory Accelerator.
//
// The register-line pass B of fft_fast.cuh (k_fr_mid) is bound by latency, not by DRAM, the FP64 pipe or shared memory
// (ncu, profiles/r01_ncu_full_summary.txt: DRAM 21 %, FP64 36 %, issue active 26 % at 7 warps per SM): a CTA loads its
// tile with 32 dependent-latency global loads per thread, transforms it, stores it, and nothing overlaps the three.
// Here one persistent CTA per SM walks over its tiles and the NEXT tile is always in flight: one elected thread issues
// a 5-D cp.async.bulk.tensor (box = 2^LGC x0 sites x all of x2 x all of x3 of one component and one x1) into the other
// of two staging buffers and arms an mbarrier with the byte count; the copy costs neither registers nor issue slots
// and completes on the barrier while all warps transform the current tile.  Phase 1 reads its axis-2 lines from the
// (dense) staging buffer and writes the padded work tile; phases 2 and 3 are those of k_fr_mid; phase 3 stores straight
// from registers (plain stores retire asynchronously).  Same arithmetic, same stored order, same results as k_fr_mid.
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

// Geometry of a pass-B tile: staging buffer dense [i3][i2][i0] (what the TMA box writes), work tile padded as MidGeom.
template <int LG2, int LG3, int LGC> struct TmaMidGeom {
    using MG = MidGeom<LG2, LGC>;
    static constexpr int L2 = 1 << LG2, L3 = 1 << LG3, C0 = 1 << LGC;
    static constexpr int TILE = C0 * L2 * L3;                       // complex numbers per tile
    static constexpr unsigned TILE_BYTES = TILE * sizeof(cplx);
    static constexpr int WORK = MG::S2 * L3;
    // shared memory: two staging buffers, the work tile, the p^2 tables of axes 2,3
    // (+ slack: the kernel rounds the dynamic shared-memory base up to the 128 bytes a TMA destination needs)
    static constexpr size_t SMEM = (size_t)(2 * TILE + WORK) * sizeof(cplx) + (size_t)(L2 + L3) * 8 + 128;
};

#ifndef LGF_TB_NT
#define LGF_TB_NT 128
#endif

// The field as a 5-D tensor of reals for the TMA unit: (2 L0 reals, L1, L2, L3, 4 components); a pass-B tile is the box
// (2 C0, 1, L2, L3, 1) at (2 C0 chunk, x1, 0, 0, comp).  n_tiles = 4 L1 (L0 / C0); tile index = chunk + nChunks (x1 + L1 comp).
template <int LG2, int LG3, int LGC, int NT>
__global__ void __launch_bounds__(NT, 1) k_tb_mid(const __grid_constant__ CUtensorMap tmap, cplx* __restrict__ field, Geom G, FftTables T,
                                                  double scale, Ctl* ctl, const double2* partials, FinArgs fa, int n_tiles) {
    pdl_enter();
    __shared__ int s_done;
    __shared__ __align__(8) uint64_t full[2];
    pass_b_entry<NT>(partials, fa, ctl, &s_done);
    using TG = TmaMidGeom<LG2, LG3, LGC>;
    using MG = MidGeom<LG2, LGC>;
    constexpr int L2 = TG::L2, L3 = TG::L3, C0 = TG::C0, S1 = MG::S1, S2 = MG::S2, TILE = TG::TILE;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // a TMA destination must be 128-byte aligned; the dynamic shared memory starts behind the static variables
    cplx* stage = reinterpret_cast<cplx*>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));      // [2][TILE]
    cplx* work = stage + 2 * TILE;
    double* s2 = reinterpret_cast<double*>(work + TG::WORK);
    double* s3 = s2 + L2;
    for (int i = threadIdx.x; i < L2; i += NT) s2[i] = T.s[2][i];
    for (int i = threadIdx.x; i < L3; i += NT) s3[i] = T.s[3][i];
    const int lgChunks = G.lg[0] - LGC;
    auto issue = [&](int tile, int buf) {                              // one thread: arm the barrier, start the copy
        const int chunk = tile & ((1 << lgChunks) - 1);
        const int x1 = (tile >> lgChunks) & (G.L[1] - 1);
        const int comp = tile >> (lgChunks + G.lg[1]);
        mbar_expect_tx(&full[buf], TG::TILE_BYTES);
        tma_load_5d(stage + buf * TILE, &tmap, &full[buf], chunk << (LGC + 1), x1, 0, 0, comp);
    };
    int tile = blockIdx.x;
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1); mbar_init(&full[1], 1);
        mbar_init_fence();
        // a copy in flight must never outlive its CTA: nothing is issued when the run is already over
        if (!s_done && tile < n_tiles) issue(tile, 0);
    }
    __syncthreads();
    if (s_done) return;                                  // one reading per CTA, behind a barrier (pass_b_entry)
    const int sh2 = G.sh[2], sh3 = G.sh[3];
#pragma unroll 1
    for (int it = 0; tile < n_tiles; it++, tile += gridDim.x) {
        const int buf = it & 1;
        // the other staging buffer was last read in phase 1 of the previous tile, two barriers ago
        if (threadIdx.x == 0 && tile + (int)gridDim.x < n_tiles) issue(tile + gridDim.x, buf ^ 1);
        const int chunk = tile & ((1 << lgChunks) - 1);
        const int x1 = (tile >> lgChunks) & (G.L[1] - 1);
        const int comp = tile >> (lgChunks + G.lg[1]);
        cplx* gbase = field + (long long)comp * G.V + (chunk << LGC) + ((long long)x1 << G.sh[1]);
        const cplx* st = stage + buf * TILE;
        mbar_wait(&full[buf], (it >> 1) & 1);
        // phase 1: lines along axis 2, one per (i0, i3), from the staging buffer: forward -> work tile
#pragma unroll 1
        for (int ln = threadIdx.x; ln < C0 * L3; ln += NT) {
            const int i0 = ln % C0, i3 = ln / C0;
            const cplx* q = st + i0 + i3 * (C0 * L2);
            cplx v[L2];
#pragma unroll
            for (int m = 0; m < L2; m++) v[m] = q[m * C0];
            line_fft<LG2, false, false>(v);
            cplx* p = work + i0 + i3 * S2;
#pragma unroll
            for (int m = 0; m < L2; m++) p[m * S1] = v[m];
        }
        __syncthreads();
        // phase 2: lines along axis 3, one per (i0, i2): forward, filter X~ = (p2max / (V p2)) Delta~ at the stored
        // positions (zero mode -> 0), inverse                                                       [north_star step 2]
#pragma unroll 1
        for (int ln = threadIdx.x; ln < C0 * L2; ln += NT) {
            const int i0 = ln % C0, i2 = ln / C0;
            cplx* p = work + i0 + i2 * S1;
            cplx v[L3];
#pragma unroll
            for (int m = 0; m < L3; m++) v[m] = p[m * S2];
            line_fft<LG3, true, false>(v);
            const double s012 = T.s[0][(chunk << LGC) + i0] + T.s[1][x1] + s2[i2];
#pragma unroll
            for (int m = 0; m < L3; m++) {
                const double p2 = s012 + s3[m];
                v[m] = cscale(v[m], (real)((p2 > 0.0) ? scale / p2 : 0.0));
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
            const cplx* p = work + i0 + i3 * S2;
            cplx v[L2];
#pragma unroll
            for (int m = 0; m < L2; m++) v[m] = p[m * S1];
            line_fft<LG2, false, true>(v);
            cplx* gq = gbase + i0 + ((long long)i3 << sh3);
#pragma unroll
            for (int m = 0; m < L2; m++) st_field(gq + ((long long)m << sh2), v[m]);
        }
        __syncthreads();                                 // the work tile is rewritten by the next tile's phase 1
    }
}

}  // namespace lgf
