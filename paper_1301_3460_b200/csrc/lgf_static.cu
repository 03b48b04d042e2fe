// lgf_static.cu -- lgf_measure_static: theta and F of a gauge configuration from a call that allocates nothing.
//
// Who this is for.  The context calls (lgf_create, lgf_scan_alpha, ...) obtain device memory with cudaMalloc.  Some
// programs that want to watch theta and F of their links cannot afford that:
//   * a Monte Carlo production job whose own pool has taken all of the HBM at start-up: a cudaMalloc from a library
//     finds nothing left and fails, although the job has plenty of memory in its pool;
//   * a program inside a framework with a caching allocator (PyTorch): memory the framework has cached is invisible to
//     cudaMalloc, so a library allocation can run out of memory, or push the framework into it later;
//   * a measurement hook inside a running update loop: cudaMalloc and cudaFree synchronise the whole device, so each
//     call would stall every other stream of the job for the length of its queue.
// For them S1's lattice sums are offered as one stateless entry point.  The caller passes the links (DEVICE, canonical
// order) and a DEVICE buffer for the two results; the block partials -- the one piece of scratch memory the step
// needs -- live in a file-scope __device__ array that is part of the loaded library image.
//
// The kernel is a variant of k_delta (kernels.cuh): same per-site arithmetic in the same order, same 128-site blocks,
// same fixed-order final sum as k_finalize; it reads the canonical [V][4][3][3] array instead of the context's
// structure-of-arrays store, writes no Delta field, and works for any extents (not only powers of two).
//
// What a user has to know:
//   * The array costs LGF_STATIC_MAX_SITES / 128 * 16 B = 2 MiB on every GPU of the process that loads the library,
//     from load to exit, whether or not the call is ever made.
//   * Lattices of more than LGF_STATIC_MAX_SITES sites are refused (LGF_ERR_UNSUPPORTED, text in
//     lgf_measure_static_error()); nothing is launched.
//   * The first call on each device looks up the array's device address (cudaGetSymbolAddress) and keeps it; that
//     first call should be made before any stream capture is begun.  Later calls only launch two kernels.
//   * The array is shared by every call on that device and keeps what the last call left in it.  The second kernel
//     reads exactly the n_blocks entries the first kernel of the same call wrote, so nothing has to be cleared and
//     stale entries are never read -- but two calls that overlap on the GPU (different streams, or different host
//     threads on different streams) write the same entries and race.  Order them on one stream or with events.
//   * No cudaMalloc, cudaFree, cudaMallocHost, stream or event creation, no library routine that allocates.
#include "../../include/lgf.h"
#include "su3.cuh"

#include <cstdio>
#include <mutex>

constexpr int ST_BLOCK = 128;                                          // sites per block, as k_delta
constexpr long long ST_MAX_BLOCKS = LGF_STATIC_MAX_SITES / ST_BLOCK;   // 131072 partials = 2 MiB
constexpr int ST_MAX_DEVICES = 64;

// The scratch memory: one (theta part, F part) pair per 128-site block.  In host code this name is only a handle for
// cudaGetSymbolAddress (scratch_address below), never an address to hand to a kernel.
static __device__ __align__(256) double2 g_static_partials[ST_MAX_BLOCKS];

namespace {

using lgf::cplx;
using lgf::mk;
using lgf::cnorm2;

std::mutex g_setup_lock;
double2* g_partials_ptr[ST_MAX_DEVICES];     // device address of g_static_partials on device i, once looked up
thread_local char g_err[256] = "";

struct StaticGeom {
    int L[4];
    long long stride[4];     // site-index stride of axis mu
    long long V;
};

// One link of the canonical array: 9 consecutive complex doubles at (x*4 + mu)*9.
__device__ __forceinline__ void load_link_aos(const double2* __restrict__ links, long long x, int mu, cplx (&u)[9]) {
    const double2* p = links + (x * 4 + mu) * 9;
#pragma unroll
    for (int c = 0; c < 9; c++) u[c] = __ldg(p + c);
}

// As acc_link of kernels.cuh: the independent entries of A - A^dag, A accumulating sg * U.
__device__ __forceinline__ void acc_link(const cplx (&u)[9], double sg, cplx& d01, cplx& d02, cplx& d12, double& i0, double& i1, double& i2) {
    d01.x = fma(sg, u[1].x - u[3].x, d01.x); d01.y = fma(sg, u[1].y + u[3].y, d01.y);
    d02.x = fma(sg, u[2].x - u[6].x, d02.x); d02.y = fma(sg, u[2].y + u[6].y, d02.y);
    d12.x = fma(sg, u[5].x - u[7].x, d12.x); d12.y = fma(sg, u[5].y + u[7].y, d12.y);
    i0 = fma(sg, u[0].y, i0); i1 = fma(sg, u[4].y, i1); i2 = fma(sg, u[8].y, i2);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// Block sum of two values in a fixed order; result in thread 0.  red: 64 doubles of shared memory.
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

// S1 without the Delta store: per site Tr[Delta Delta^dag] and sum_mu Re Tr U_mu(x), summed over the block's 128 sites
// into partials[blockIdx.x] = (theta part, F part).  Sites beyond V (last block of a lattice whose volume is not a
// multiple of 128) contribute zeros.
__global__ void __launch_bounds__(ST_BLOCK) k_delta_static(const double2* __restrict__ links, double2* __restrict__ partials, StaticGeom G) {
    __shared__ double red[64];
    const long long x = (long long)blockIdx.x * ST_BLOCK + threadIdx.x;
    double th = 0.0, fs = 0.0;
    if (x < G.V) {
        cplx d01 = mk(0, 0), d02 = mk(0, 0), d12 = mk(0, 0);
        double i0 = 0, i1 = 0, i2 = 0, retr = 0;
        long long rest = x;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const int xm = (int)(rest % G.L[mu]);
            rest /= G.L[mu];
            const long long xb = (xm == 0) ? x + (long long)(G.L[mu] - 1) * G.stride[mu] : x - G.stride[mu];
            cplx u[9];
            load_link_aos(links, x, mu, u);
            retr += u[0].x + u[4].x + u[8].x;
            acc_link(u, -1.0, d01, d02, d12, i0, i1, i2);
            load_link_aos(links, xb, mu, u);
            acc_link(u, 1.0, d01, d02, d12, i0, i1, i2);
        }
        const double tr3 = (2.0 / 3.0) * (i0 + i1 + i2);
        const double e0 = 2.0 * i0 - tr3, e1 = 2.0 * i1 - tr3, e2 = 2.0 * i2 - tr3;
        th = 2.0 * (cnorm2(d01) + cnorm2(d02) + cnorm2(d12)) + e0 * e0 + e1 * e1 + e2 * e2;
        fs = retr;
    }
    block_sum2(th, fs, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(th, fs);
}

// One block: the n partials in a fixed order (strided per thread, then the tree), as k_finalize; out = (F, theta).
__global__ void __launch_bounds__(1024) k_sum_static(const double2* __restrict__ partials, int n, double* __restrict__ out, double inv3V, double inv12V) {
    __shared__ double red[64];
    double a = 0, b = 0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) { double2 p = partials[i]; a += p.x; b += p.y; }
    block_sum2(a, b, red);
    if (threadIdx.x == 0) { out[0] = b * inv12V; out[1] = a * inv3V; }
}

// Device address of the scratch array on the current device, looked up on first use.
lgf_status scratch_address(double2** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        snprintf(g_err, sizeof g_err, "lgf_measure_static: cudaGetDevice -> %s", cudaGetErrorString(e));
        cudaGetLastError();
        return LGF_ERR_CUDA;
    }
    if (dev < 0 || dev >= ST_MAX_DEVICES) {
        snprintf(g_err, sizeof g_err, "lgf_measure_static: device ordinal %d outside 0..%d", dev, ST_MAX_DEVICES - 1);
        return LGF_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_partials_ptr[dev]) {
        double2* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_static_partials);
        if (e != cudaSuccess || !p) {
            snprintf(g_err, sizeof g_err, "lgf_measure_static: cudaGetSymbolAddress on device %d -> %s", dev, cudaGetErrorString(e));
            cudaGetLastError();
            return LGF_ERR_CUDA;
        }
        g_partials_ptr[dev] = p;
    }
    *out = g_partials_ptr[dev];
    return LGF_OK;
}

}  // namespace

extern "C" {

lgf_status lgf_measure_static(const double* dev_links, const int dims[4], void* cuda_stream, double* dev_out) {
    g_err[0] = 0;
    if (!dev_links || !dims || !dev_out) {
        snprintf(g_err, sizeof g_err, "lgf_measure_static: NULL argument");
        return LGF_ERR_INVALID_ARG;
    }
    StaticGeom G;
    long long V = 1;
    for (int mu = 0; mu < 4; mu++) {
        if (dims[mu] < 1) {
            snprintf(g_err, sizeof g_err, "lgf_measure_static: extent L%d = %d", mu, dims[mu]);
            return LGF_ERR_INVALID_ARG;
        }
        G.L[mu] = dims[mu];
        G.stride[mu] = V;
        V *= dims[mu];
        if (V > (long long)LGF_STATIC_MAX_SITES) {
            snprintf(g_err, sizeof g_err, "lgf_measure_static: lattice %dx%dx%dx%d has more than LGF_STATIC_MAX_SITES = %lld sites "
                     "(the static scratch array holds one partial sum per 128 sites)", dims[0], dims[1], dims[2], dims[3], (long long)LGF_STATIC_MAX_SITES);
            return LGF_ERR_UNSUPPORTED;
        }
    }
    G.V = V;
    double2* partials = nullptr;
    lgf_status st = scratch_address(&partials);
    if (st != LGF_OK) return st;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    const int n_blocks = (int)((V + ST_BLOCK - 1) / ST_BLOCK);
    k_delta_static<<<(unsigned)n_blocks, ST_BLOCK, 0, stream>>>(reinterpret_cast<const double2*>(dev_links), partials, G);
    k_sum_static<<<1, n_blocks > 8192 ? 1024 : 256, 0, stream>>>(partials, n_blocks, dev_out, 1.0 / (3.0 * (double)V), 1.0 / (12.0 * (double)V));
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(g_err, sizeof g_err, "lgf_measure_static: launch -> %s", cudaGetErrorString(e));
        return LGF_ERR_CUDA;
    }
    return LGF_OK;
}

const char* lgf_measure_static_error(void) { return g_err; }

}  // extern "C"
