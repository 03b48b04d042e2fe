// lgf_api.cu -- host side of the C ABI declared in include/lgf.h: context, workspace carving, FFT tables,
// the iteration driver (device-side stop flag, CUDA-graph replay) and the boundary copies.
// There is deliberately no CPU fallback: every compute entry point needs a CUDA device.
#include "../../include/lgf.h"

// This file is compiled twice into liblgf.so: as it stands (fp64: real = double) and with -DLGF_F32 (fp32 storage and
// arithmetic: real = float, lattice sums still double).  The fp32 build lives in its own namespace, has its own
// context type and exports its entry points as lgf32_*; the fp64 entry points (the public lgf_* names) forward to
// them when the context, or the precision argument of lgf_create*, says LGF_FP32.  Every context starts with its
// precision, so the public opaque handle can be told apart.
#ifdef LGF_F32
#define lgf lgf32
#define lgf_ctx lgf32_ctx
#define lgf_workspace_bytes lgf32_workspace_bytes
#define lgf_create_ex lgf32_create_ex
#define lgf_create lgf32_create
#define lgf_destroy lgf32_destroy
#define lgf_load_links_device lgf32_load_links_device
#define lgf_load_links lgf32_load_links
#define lgf_get_links_device lgf32_get_links_device
#define lgf_get_links lgf32_get_links
#define lgf_load_links_12 lgf32_load_links_12
#define lgf_get_links_12 lgf32_get_links_12
#define lgf_iterate lgf32_iterate
#define lgf_fix lgf32_fix
#define lgf_measure lgf32_measure
#define lgf_scan_alpha lgf32_scan_alpha
#define lgf_get_history lgf32_get_history
#define lgf_get_field lgf32_get_field
#define lgf_set_option lgf32_set_option
#define lgf_get_option lgf32_get_option
#define lgf_set_profiling lgf32_set_profiling
#define lgf_get_profile lgf32_get_profile
#define lgf_launch_count lgf32_launch_count
#define lgf_last_error lgf32_last_error
struct lgf_ctx;
extern "C" void lgf_destroy(lgf_ctx* c);
#define LGF_THIS_PREC LGF_FP32
#define FWD32(call)
#define FWD32V(call)
#else
#define LGF_THIS_PREC LGF_FP64
extern "C" {
size_t lgf32_workspace_bytes(const int dims[4], lgf_precision p, lgf_storage s);
lgf_status lgf32_create(const int dims[4], lgf_precision p, lgf_storage s, lgf_ctx** out);
lgf_status lgf32_create_ex(const int dims[4], lgf_precision p, lgf_storage s, void* ws, size_t bytes, void* stream, lgf_ctx** out);
void lgf32_destroy(lgf_ctx* c);
lgf_status lgf32_load_links(lgf_ctx* c, const double* host_links);
lgf_status lgf32_load_links_device(lgf_ctx* c, const double* dev_links);
lgf_status lgf32_get_links(lgf_ctx* c, double* host_links);
lgf_status lgf32_load_links_12(lgf_ctx* c, const double* host_rows);
lgf_status lgf32_get_links_12(lgf_ctx* c, double* host_rows);
lgf_status lgf32_get_links_device(lgf_ctx* c, double* dev_links);
lgf_status lgf32_iterate(lgf_ctx* c, int n, double alpha, double* F, double* theta);
lgf_status lgf32_fix(lgf_ctx* c, double alpha, double theta_tol, int max_iter, int* n_iter, double* F, double* theta);
lgf_status lgf32_measure(lgf_ctx* c, double* F, double* theta, double* plaq);
lgf_status lgf32_scan_alpha(lgf_ctx* c, const double* alphas, int n, double theta_tol, int max_iter, int* counts, double* F_final, int* best);
lgf_status lgf32_get_history(lgf_ctx* c, double* hist, int capacity, int* n_out);
lgf_status lgf32_get_field(lgf_ctx* c, lgf_field which, double alpha, double* host_field);
lgf_status lgf32_set_option(lgf_ctx* c, lgf_option opt, int value);
lgf_status lgf32_get_option(lgf_ctx* c, lgf_option opt, int* value);
lgf_status lgf32_set_profiling(lgf_ctx* c, int on);
lgf_status lgf32_get_profile(lgf_ctx* c, double ms[LGF_MAX_KERNELS], long long n[LGF_MAX_KERNELS]);
long long lgf32_launch_count(lgf_ctx* c);
const char* lgf32_last_error(lgf_ctx* c);
// mixed precision (internal, not in lgf.h): start an fp32 phase on links the caller writes to the returned device
// buffer (float2 SoA, same order as the fp64 store) with the accumulated transformation reset to 1; and read it back
void* lgf32_x_begin(lgf_ctx* c);
void* lgf32_x_gacc(lgf_ctx* c);
}
// forward to the fp32 twin when the context is an fp32 one (the precision is the first member of both context types)
#define FWD32(call) if (c && *reinterpret_cast<const int*>(c) == (int)LGF_FP32) return call;
#define FWD32V(call) if (c && *reinterpret_cast<const int*>(c) == (int)LGF_FP32) { call; return; }
#endif

#include "kernels.cuh"
#include "fft_fast.cuh"
#include "fft_tma.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace lgf;

namespace {

enum KernelSlot {
    K_DELTA = 0, K_FFT01_FWD, K_FFT01_DELTA_FWD, K_FINALIZE, K_FFT23_MID, K_FFT01_INV, K_FFT01_INV_G, K_UPDATE_G,
    K_LAYOUT_IN, K_LAYOUT_OUT, K_PLAQUETTE, K_MISC, K_FA_DELTA_FWD, K_FA_MID, K_FA_INV, K_FA_INV_G,
    K_UPDATE_QUAD, K_FA_FWD1, K_FA_INV1, K_FR_MID, K_CL_DELTA_FWD, K_TB_MID, K_TM_MID, K_TA_DELTA_FWD, K_TR_MID, K_NSLOTS
};
static_assert(K_NSLOTS <= LGF_MAX_KERNELS, "kernel slot table");
const char* const kKernelNames[LGF_MAX_KERNELS] = {
    "k_delta", "k_fft01_fwd", "k_fft01_delta_fwd", "k_finalize", "k_fft23_mid", "k_fft01_inv", "k_fft01_inv_g", "k_update_g",
    "k_layout_in", "k_layout_out", "k_plaquette", "misc", "k_fa_delta_fwd", "k_fa_mid", "k_fa_inv", "k_fa_inv_g",
    "k_update_quad", "k_fa_fwd1", "k_fa_inv1", "k_fr_mid", "k_cl_delta_fwd", "k_tb_mid", "k_tm_mid", "k_ta_delta_fwd", "k_tr_mid"};

constexpr int HIST_CAP = 1 << 16;
// mixed precision: the fp32 phase ends when theta has not halved within this many iterations (a rough thermalised
// configuration at beta = 5.7 halves theta every ~30 iterations at alpha = 0.08; a wrong "stalled" only hands over early)
#ifndef LGF_MIXED_STALL_WINDOW
#define LGF_MIXED_STALL_WINDOW 256
#endif
constexpr long long STAGE_SITES = 1 << 17;   // sites per staging chunk of the boundary copies
constexpr int MAX_SMEM = 200 * 1024;

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {   // offsets into the workspace
    size_t links, field, gbuf, partials, ctl, hist, tables, scratch, staging, total;
    int n_partials;
    long long stage_sites;
};

bool dims_ok(const int dims[4], int lg[4]) {
    for (int k = 0; k < 4; k++) {
        int L = dims[k];
        if (L < 4 || L > 128 || (L & (L - 1))) return false;
        int l = 0; while ((1 << l) < L) l++;
        lg[k] = l;
    }
    if ((long long)dims[0] * dims[1] > 4096 || (long long)dims[2] * dims[3] > 4096) return false;
    return true;
}

Layout make_layout(const int dims[4], int NC) {
    Layout o;
    const long long V = (long long)dims[0] * dims[1] * dims[2] * dims[3];
    size_t off = 0;
    o.links = off; off = align_up(off + (size_t)V * 4 * NC * sizeof(cplx), 256);
    o.field = off; off = align_up(off + (size_t)V * 4 * sizeof(cplx), 256);
    o.gbuf = off; off = align_up(off + (size_t)V * 6 * sizeof(cplx), 256);
    o.n_partials = (int)(V / 128);                       // k_delta / k_plaquette: one per 128-site block
    if (o.n_partials < dims[2] * dims[3]) o.n_partials = dims[2] * dims[3];   // fused pass A: one per (x2,x3) plane
    o.partials = off; off = align_up(off + (size_t)o.n_partials * 16, 256);
    o.ctl = off; off = align_up(off + sizeof(Ctl), 256);
    o.hist = off; off = align_up(off + (size_t)HIST_CAP * 16, 256);
    o.tables = off; off = align_up(off + 4 * 128 * 16 + 4 * 128 * 8, 256);
    o.scratch = off; off = align_up(off + 256, 256);
    o.stage_sites = V < STAGE_SITES ? V : STAGE_SITES;
    o.staging = off; off = align_up(off + (size_t)o.stage_sites * 4 * 9 * 16, 256);
    o.total = off;
    return o;
}

// Stage radices of an axis of length 2^lgL; b_axis: axes 1 and 3 (see fft_tile.cuh); mid: axes 2,3 (pass B), whose
// 64-point plan is [4,4,4] -- the stored order of the 16 x 4 / 4 x 16 stages of the compile-time-sized pass B (PlanM).
AxisPlan make_plan(int lgL, bool b_axis, bool mid) {
    AxisPlan p; p.nst = 0; p.lgr[0] = p.lgr[1] = p.lgr[2] = 0;
    if (lgL == 5 && b_axis) { p.nst = 2; p.lgr[0] = 2; p.lgr[1] = 3; return p; }
    if (lgL == 6 && mid) { p.nst = 3; p.lgr[0] = p.lgr[1] = p.lgr[2] = 2; return p; }
    int lgN = lgL;
    while (lgN > 0) {
        const int lgR = (lgN == 1) ? 1 : ((lgN == 2 || lgN == 4) ? 2 : 3);
        p.lgr[p.nst++] = lgR;
        lgN -= lgR;
    }
    return p;
}

// frequency index held at stored position p after the forward DIF stages of fft_tile.cuh
int stored_freq(int p, int lgL, const AxisPlan& plan) {
    int n = 0, mult = 1, lgN = lgL;
    for (int k = 0; k < plan.nst; k++) {
        const int lgR = plan.lgr[k];
        const int lgs = lgN - lgR;
        const int m = p >> lgs;
        p &= (1 << lgs) - 1;
        n += m * mult;
        mult <<= lgR;
        lgN -= lgR;
    }
    return n;
}

}  // namespace

struct lgf_ctx {
    int precision;          // LGF_FP64 or LGF_FP32: FIRST member of the context in both builds
    Geom G;
    int NC;                 // 6 or 9
    Layout lay;
    char* ws;               // workspace base (device)
    bool own_ws, own_stream;
    cudaStream_t stream;
    cudaStream_t copy_stream;           // boundary copies (overlap with the layout kernels on `stream`)
    cudaEvent_t ev_copy[2], ev_kern[2]; // per staging half: copy done / layout kernel done
    cplx *links, *field, *gbuf;
    dcplx* staging;         // host-facing double complex (AoS chunks of the boundary copies)
    double2 *partials, *hist;
    Ctl* ctl;
    FftTables T;
    Ctl* h_ctl;             // pinned
    bool loaded;
    // mixed precision: the fp64 context owns an fp32 shadow context (same stream); the fp32 context accumulates G
    lgf_ctx* shadow;        // fp64 build: opaque fp32 context, or nullptr
    char* shadow_ws;        // its workspace when this context allocated it
    int acc_g;              // fp32 build: the update also accumulates Gacc(x) <- g(x) Gacc(x) in gbuf
    int mixed_n32;          // fp32 iterations of the last mixed lgf_fix
    int mixed_switch;       // the fp32 phase aims at theta = 10^-mixed_switch (LGF_OPT_MIXED_SWITCH)
    int stall_window;       // fp32 build, mixed precision: stagnation guard of the fp32 phase (Ctl::stall_window), 0 = off
    int pending_np;         // S5 inside pass B: partials of the S1 just enqueued that no k_finalize has reduced yet
    // options (include/lgf.h lgf_option)
    int opt_store_g, opt_graph, opt_batch, opt_fast, opt_pdl, opt_accel, opt_tma;
    // pass B on TMA-staged tiles (fft_tma.cuh): the field as a 5-D tensor map, whether it could be built
    CUtensorMap tm_field, tm_field_half;
    bool tma_b, ring_b;
    LinkMaps tm_links;      // pass A with the links staged by the TMA unit (k_ta_delta_fwd)
    bool tma_a;
    int sms;                // SMs of the device
    // compile-time-sized FFT passes available for this lattice: pass A (fused Delta), B (middle), C (inverse)
    bool fast_a, fast_b, fast_c, big_p, cl_ok;
    size_t smem_fa, smem_fb, smem_fc, smem_p1, smem_cl;
    int fb_lgC;
    // derived launch parameters of the generic passes
    int fft01_ncomp_fused_ok, fft01_ncomp, fft01_threads, fft23_lgC, fft23_S1, fft23_S2, fft23_threads;
    size_t smem01_fused, smem01, smem23;
    // graph cache: the executable graph of opt_batch iteration bodies and the full selection it was captured with
    struct GraphKey { double half_alpha; int nb, nd, acc_g, store_g, fast, pdl, accel, tma; };
    cudaGraphExec_t graph_exec;
    GraphKey graph_key;
    // profiling
    int profiling;
    cudaEvent_t ev0, ev1;
    std::vector<cudaEvent_t> ev_pool;   // profiling: event pairs recorded around launches, resolved in batches
    std::vector<int> ev_slot;           // kernel slot of each recorded pair
    double prof_ms[LGF_MAX_KERNELS];
    long long prof_n[LGF_MAX_KERNELS];
    long long launches;
    std::string err;
    bool capturing;
};

namespace {

#define CK(call)                                                                                           \
    do {                                                                                                   \
        cudaError_t e_ = (call);                                                                           \
        if (e_ != cudaSuccess) {                                                                           \
            char b_[512];                                                                                  \
            snprintf(b_, sizeof b_, "%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            c->err = b_;                                                                                   \
            return LGF_ERR_CUDA;                                                                           \
        }                                                                                                  \
    } while (0)

// Profiling: resolve the event pairs recorded so far (one synchronisation for the whole batch, so the kernels run
// back to back on the device and the pairs measure device time, not launch latency).
constexpr size_t PROF_PAIRS = 1024;
void prof_flush(lgf_ctx* c) {
    if (c->ev_slot.empty()) return;
    cudaStreamSynchronize(c->stream);
    for (size_t i = 0; i < c->ev_slot.size(); i++) {
        float ms = 0;
        if (cudaEventElapsedTime(&ms, c->ev_pool[2 * i], c->ev_pool[2 * i + 1]) == cudaSuccess) {
            c->prof_ms[c->ev_slot[i]] += ms; c->prof_n[c->ev_slot[i]]++;
        }
    }
    c->ev_slot.clear();
}
// Launch bookkeeping: counts every kernel; in profiling mode brackets it with a pair of events.
struct LaunchScope {
    lgf_ctx* c; int slot; bool rec;
    LaunchScope(lgf_ctx* c_, int s) : c(c_), slot(s), rec(false) {
        if (c->profiling && !c->capturing) {
            if (c->ev_slot.size() >= PROF_PAIRS) prof_flush(c);
            const size_t i = c->ev_slot.size();
            while (c->ev_pool.size() < 2 * (i + 1)) { cudaEvent_t e = nullptr; if (cudaEventCreate(&e) != cudaSuccess) return; c->ev_pool.push_back(e); }
            cudaEventRecord(c->ev_pool[2 * i], c->stream);
            rec = true;
        }
    }
    ~LaunchScope() {
        if (!c->capturing) c->launches++;
        if (rec) {
            cudaEventRecord(c->ev_pool[2 * c->ev_slot.size() + 1], c->stream);
            c->ev_slot.push_back(slot);
        }
    }
};

// Launch of an iteration-body kernel: with opt_pdl the launch carries the programmatic-stream-serialization attribute
// (the kernels call pdl_enter(), su3.cuh); stream capture turns it into a programmatic graph edge.
template <typename... KArgs, typename... Args>
void launch_k(lgf_ctx* c, void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = c->opt_pdl ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// Opt a kernel in to large dynamic shared memory.  The attribute is a per-function CAP shared by every context in the
// process, so it is always raised to the device's opt-in maximum -- setting it to one context's tile size would lower it
// under the feet of another live context with a larger lattice.
template <typename K> cudaError_t set_smem(K kern, size_t bytes) {
    static int optin = 0;
    if (!optin) {
        int dev = 0;
        cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess || optin <= 0) { optin = 0; return cudaErrorInvalidValue; }
    }
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, kern);
    if (e != cudaSuccess) return e;
    const long long cap = (long long)optin - (long long)fa.sharedSizeBytes;      // static + dynamic <= the opt-in maximum
    if (cap < (long long)bytes) return cudaErrorInvalidValue;
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cap);
}

// ---- compile-time-sized FFT passes (fft_fast.cuh): the lattices they cover, and their launchers ----------------
constexpr int FAD_NT = 256;           // threads per CTA of pass A (k_fa_delta_fwd)
constexpr int FC_NT = 256;            // threads per CTA of pass C (k_fa_inv) and of the one-component plane passes
constexpr int CL_NT = 512;            // threads per CTA of the CTA-pair pass A (k_cl_delta_fwd)
constexpr int FB_NT = 256;            // threads per CTA of the stage-wise pass B when its tile is below 100 KB
// (lg of the fast axis, lg of the slow axis) pairs instantiated for each pass: extents 16 and 32 ...
#define LGF_FAST_PAIRS(X) X(4, 4) X(4, 5) X(5, 4) X(5, 5)
// ... and pairs with a 64 extent: the (x0,x1) plane passes take one component per CTA (four 64-wide tiles do not fit
// one SM; 64 x 64 planes run S1 on CTA pairs, the others keep S1 a separate kernel), the (x2,x3) pass takes a shorter
// x0 chunk
#define LGF_BIG_PAIRS(X) X(5, 6) X(6, 5) X(6, 6)
// ... of which the 64-extent pass B also runs as a ring of half-chunk tiles (k_tr_mid)
#define LGF_RING_PAIRS(X) X(5, 6) X(6, 5)
// x0 chunk of pass B (2^lgC sites): tile = 2^(lga+lgb+lgC) * 16 B
constexpr int fast_mid_lgC(int lga, int lgb) { return (lga + lgb <= 9) ? 3 : ((lga + lgb == 10) ? 2 : ((lga + lgb == 11) ? 2 : 1)); }
// threads per CTA of the stage-wise pass B: one 512-thread CTA per SM when the tile is above 100 KB, else 2 x 256
constexpr int fast_mid_nt(int lga, int lgb) { return ((16 << (lga + lgb + fast_mid_lgC(lga, lgb))) > 100 * 1024) ? 512 : FB_NT; }
bool fast_pair(int lga, int lgb) {
#define X(A, B) if (lga == A && lgb == B) return true;
    LGF_FAST_PAIRS(X)
#undef X
    return false;
}
bool big_pair(int lga, int lgb) {
#define X(A, B) if (lga == A && lgb == B) return true;
    LGF_BIG_PAIRS(X)
#undef X
    return false;
}
size_t smem_fast_plane(int lga, int lgb, int ncomp) { return (size_t)(((1 << lga) + 1) * (1 << lgb) * ncomp + (1 << lga) + (1 << lgb)) * sizeof(cplx); }
size_t smem_fast_mid(int lga, int lgb, int lgC) {
    const int C0 = 1 << lgC, S2 = C0 * (1 << lga) + (C0 < 8 ? C0 : 0);
    return (size_t)(S2 * (1 << lgb) + (1 << lga) + (1 << lgb)) * sizeof(cplx) + (size_t)((1 << lga) + (1 << lgb)) * 8;
}

template <int NC> void launch_fa_delta_fwd(lgf_ctx* c) {
    LaunchScope ls(c, K_FA_DELTA_FWD);
    const unsigned grid = (unsigned)(c->G.L[2] * c->G.L[3]);
#define X(A, B) if (c->G.lg[0] == A && c->G.lg[1] == B) \
        launch_k(c, k_fa_delta_fwd<A, B, NC, FAD_NT>, grid, FAD_NT, c->smem_fa, c->links, c->field, c->partials, c->G, c->T, c->ctl);
    LGF_FAST_PAIRS(X)
#undef X
}
void launch_fa_inv(lgf_ctx* c) {
    LaunchScope ls(c, K_FA_INV);
    const unsigned grid = (unsigned)(c->G.L[2] * c->G.L[3]);
#define X(A, B) if (c->G.lg[0] == A && c->G.lg[1] == B) \
        launch_k(c, k_fa_inv<A, B, 4, FC_NT, false>, grid, FC_NT, c->smem_fc, c->field, nullptr, 0.0, c->G, c->T, c->ctl);
    LGF_FAST_PAIRS(X)
#undef X
}
void launch_fa_inv_g(lgf_ctx* c, double half_alpha) {
    LaunchScope ls(c, K_FA_INV_G);
    const unsigned grid = (unsigned)(c->G.L[2] * c->G.L[3]);
#define X(A, B) if (c->G.lg[0] == A && c->G.lg[1] == B) \
        launch_k(c, k_fa_inv<A, B, 4, FC_NT, true>, grid, FC_NT, c->smem_fc, c->field, c->gbuf, half_alpha, c->G, c->T, c->ctl);
    LGF_FAST_PAIRS(X)
#undef X
}
// 64 x 64 planes: S1 fused into pass A on CTA pairs (clusters of 2 sharing the four component tiles over DSMEM)
template <int NC> void launch_cl_delta_fwd(lgf_ctx* c) {
    LaunchScope ls(c, K_CL_DELTA_FWD);
    const unsigned grid = (unsigned)(2 * c->G.L[2] * c->G.L[3]);
    launch_k(c, k_cl_delta_fwd<6, 6, NC, CL_NT>, grid, CL_NT, c->smem_cl, c->links, c->field, c->partials, c->G, c->T, c->ctl);
}
// planes with a 64 extent: one component per CTA
void launch_fa_fwd1(lgf_ctx* c) {
    LaunchScope ls(c, K_FA_FWD1);
    const unsigned grid = (unsigned)(4 * c->G.L[2] * c->G.L[3]);
#define X(A, B) if (c->G.lg[0] == A && c->G.lg[1] == B) \
        launch_k(c, k_fa_fwd<A, B, 1, FC_NT>, grid, FC_NT, c->smem_p1, c->field, c->G, c->T, c->ctl);
    LGF_BIG_PAIRS(X)
#undef X
}
void launch_fa_inv1(lgf_ctx* c) {
    LaunchScope ls(c, K_FA_INV1);
    const unsigned grid = (unsigned)(4 * c->G.L[2] * c->G.L[3]);
#define X(A, B) if (c->G.lg[0] == A && c->G.lg[1] == B) \
        launch_k(c, k_fa_inv<A, B, 1, FC_NT, false>, grid, FC_NT, c->smem_p1, c->field, nullptr, 0.0, c->G, c->T, c->ctl);
    LGF_BIG_PAIRS(X)
#undef X
}
// S5 inside pass B: the pending number of partials of the S1 that just ran (0: k_finalize already did it)
FinArgs pending_fin(lgf_ctx* c) {
    const FinArgs fa{c->hist, 1.0 / (3.0 * (double)c->G.V), 1.0 / (3.0 * (double)c->G.nd * (double)c->G.V), c->pending_np};
    c->pending_np = 0;
    return fa;
}
// pass B, stage-wise through shared memory: 64 extents
void launch_fa_mid(lgf_ctx* c) {
    LaunchScope ls(c, K_FA_MID);
    const unsigned grid = (unsigned)(4 * c->G.L[1] * (c->G.L[0] >> c->fb_lgC));
    const double scale = 4.0 * (double)c->G.nd / (double)c->G.V;      // p2max / V
    const FinArgs fa = pending_fin(c);
#define X(A, B) if (c->G.lg[2] == A && c->G.lg[3] == B) \
        launch_k(c, k_fa_mid<A, B, fast_mid_lgC(A, B), fast_mid_nt(A, B)>, grid, fast_mid_nt(A, B), c->smem_fb, c->field, c->G, c->T, scale, c->ctl, c->partials, fa);
    LGF_BIG_PAIRS(X)
#undef X
}
// pass B with whole lines in registers (fft_fast.cuh k_fr_mid): 16/32 extents
void launch_fr_mid(lgf_ctx* c) {
    LaunchScope ls(c, K_FR_MID);
    const unsigned grid = (unsigned)(4 * c->G.L[1] * (c->G.L[0] >> c->fb_lgC));
    const double scale = 4.0 * (double)c->G.nd / (double)c->G.V;      // p2max / V
    const FinArgs fa = pending_fin(c);
#define X(A, B) if (c->G.lg[2] == A && c->G.lg[3] == B) { \
        if (c->G.nd == 3) launch_k(c, k_fr_mid<A, B, fast_mid_lgC(A, B), LGF_FR_NT, true>, grid, LGF_FR_NT, c->smem_fb, c->field, c->G, c->T, scale, c->ctl, c->partials, fa); \
        else launch_k(c, k_fr_mid<A, B, fast_mid_lgC(A, B), LGF_FR_NT, false>, grid, LGF_FR_NT, c->smem_fb, c->field, c->G, c->T, scale, c->ctl, c->partials, fa); }
    LGF_FAST_PAIRS(X)
#undef X
}

// pass B on TMA-staged tiles (fft_tma.cuh): 16/32 extents, one persistent CTA per SM
void launch_tb_mid(lgf_ctx* c) {
    LaunchScope ls(c, K_TB_MID);
    const int n_tiles = 4 * c->G.L[1] * (c->G.L[0] >> c->fb_lgC);
    const unsigned grid = (unsigned)(n_tiles < c->sms ? n_tiles : c->sms);
    const double scale = 4.0 * (double)c->G.nd / (double)c->G.V;      // p2max / V
    const FinArgs fa = pending_fin(c);
#define X(A, B) if (c->G.lg[2] == A && c->G.lg[3] == B) \
        launch_k(c, k_tb_mid<A, B, fast_mid_lgC(A, B), LGF_TB_NT>, grid, LGF_TB_NT, TmaMidGeom<A, B, fast_mid_lgC(A, B)>::SMEM, c->tm_field, c->field, c->G, c->T, scale, c->ctl, c->partials, fa, n_tiles);
    LGF_FAST_PAIRS(X)
#undef X
}

// pass A with TMA-staged links (fft_tma.cuh k_ta_delta_fwd): 16/32 extents, one persistent CTA per SM
// (instantiated for fp64 two-row storage only: two stages of 18-real links do not fit one SM, and the fp32 build keeps
// the plain-load pass A, which measured faster there)
void launch_ta_delta_fwd(lgf_ctx* c) {
#ifndef LGF_F32
    LaunchScope ls(c, K_TA_DELTA_FWD);
    const int n_planes = c->G.L[2] * c->G.L[3];
    const unsigned grid = (unsigned)(n_planes < c->sms ? n_planes : c->sms);
#define X(A, B) if (c->G.lg[0] == A && c->G.lg[1] == B) \
        launch_k(c, k_ta_delta_fwd<A, B, 6, 256>, grid, 256, TmaPlaneGeom<A, B, 6>::SMEM, c->tm_links, c->field, c->partials, c->G, c->T, c->ctl, n_planes);
    LGF_FAST_PAIRS(X)
#undef X
#else
    (void)c;
#endif
}

// pass B on TMA-staged tiles, 64 extents: the tile goes in and out through the TMA unit (fft_tma.cuh k_tm_mid)
constexpr int TM_NT = 512;             // the ring (k_tr_mid): two groups of 256
// the single-buffered 64 x 64 pass: 256 threads with two items per thread and stage (961 against 997 us at 64^4 for 512
// threads with one: the second item's shared-memory loads overlap the first one's butterflies)
constexpr int TM1_NT = 256;
void launch_tm_mid(lgf_ctx* c) {
    LaunchScope ls(c, K_TM_MID);
    const int n_tiles = 4 * c->G.L[1] * (c->G.L[0] >> c->fb_lgC);
    const unsigned grid = (unsigned)(n_tiles < c->sms ? n_tiles : c->sms);
    const double scale = 4.0 * (double)c->G.nd / (double)c->G.V;      // p2max / V
    const FinArgs fa = pending_fin(c);
#define X(A, B) if (c->G.lg[2] == A && c->G.lg[3] == B) \
        launch_k(c, k_tm_mid<A, B, fast_mid_lgC(A, B), TM1_NT>, grid, TM1_NT, TmaBigGeom<A, B, fast_mid_lgC(A, B)>::SMEM, c->tm_field, c->field, c->G, c->T, scale, c->ctl, c->partials, fa, n_tiles);
    LGF_BIG_PAIRS(X)
#undef X
}

// ... as a ring of half-chunk tiles (fft_tma.cuh k_tr_mid)
void launch_tr_mid(lgf_ctx* c) {
    LaunchScope ls(c, K_TR_MID);
    const int n_tiles = 4 * c->G.L[1] * (c->G.L[0] >> (c->fb_lgC - 1));
    const int n_pairs = n_tiles / 2;
    const unsigned grid = (unsigned)(n_pairs < c->sms ? n_pairs : c->sms);
    const double scale = 4.0 * (double)c->G.nd / (double)c->G.V;      // p2max / V
    const FinArgs fa = pending_fin(c);
#define X(A, B) if (c->G.lg[2] == A && c->G.lg[3] == B) \
        launch_k(c, k_tr_mid<A, B, fast_mid_lgC(A, B) - 1, TM_NT>, grid, TM_NT, TmaRingGeom<A, B, fast_mid_lgC(A, B) - 1>::SMEM, c->tm_field_half, c->field, c->G, c->T, scale, c->ctl, c->partials, fa, n_tiles);
    LGF_RING_PAIRS(X)
#undef X
}

// The field as a 5-D tensor of reals (2 L0, L1, L2, L3, 4 components) with the pass-B tile as its box.  The encoder is
// a driver entry point fetched at run time, so the library does not link against libcuda.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
bool make_field_tensor_map(lgf_ctx* c, int lgC, CUtensorMap* out) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return false;
    }
    const Geom& G = c->G;
    const cuuint64_t esz = sizeof(cplx);
    const cuuint64_t dims[5] = {(cuuint64_t)2 * G.L[0], (cuuint64_t)G.L[1], (cuuint64_t)G.L[2], (cuuint64_t)G.L[3], 4};
    const cuuint64_t strides[4] = {esz * G.L[0], esz * G.L[0] * G.L[1], esz * G.L[0] * G.L[1] * G.L[2], esz * (cuuint64_t)G.V};
    const cuuint32_t box[5] = {(cuuint32_t)(2 << lgC), 1, (cuuint32_t)G.L[2], (cuuint32_t)G.L[3], 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = reinterpret_cast<EncodeTiledFn>(fn)(out, sizeof(real) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
        5, c->field, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// The link store as a 3-D tensor of reals (2 L0 L1 reals of a plane, L2 L3 planes, 4 NC streams) with the three boxes of
// a pass-A stage: 128 sites x all streams, 128 sites x the NC streams of one direction, one x0 row x NC streams.
bool make_link_tensor_maps(lgf_ctx* c) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return false;
    }
    const Geom& G = c->G;
    const cuuint64_t esz = sizeof(cplx);
    const cuuint64_t plane = (cuuint64_t)G.L[0] * G.L[1];
    const cuuint64_t dims[3] = {2 * plane, (cuuint64_t)G.L[2] * G.L[3], (cuuint64_t)(4 * c->NC)};
    const cuuint64_t strides[2] = {esz * plane, esz * (cuuint64_t)G.V};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUtensorMapDataType dt = sizeof(real) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const cuuint32_t boxes[3][3] = {{2 * TA_SS, 1, (cuuint32_t)(4 * c->NC)}, {2 * TA_SS, 1, (cuuint32_t)c->NC}, {(cuuint32_t)(2 * G.L[0]), 1, (cuuint32_t)c->NC}};
    CUtensorMap* maps[3] = {&c->tm_links.own, &c->tm_links.nb, &c->tm_links.row};
    for (int k = 0; k < 3; k++)
        if (reinterpret_cast<EncodeTiledFn>(fn)(maps[k], dt, 3, c->links, dims, strides, boxes[k], estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    return true;
}

lgf_status setup_fast(lgf_ctx* c) {
    const Geom& G = c->G;
    c->fast_a = c->fast_c = fast_pair(G.lg[0], G.lg[1]);
    c->fast_b = fast_pair(G.lg[2], G.lg[3]) || big_pair(G.lg[2], G.lg[3]);
    c->big_p = big_pair(G.lg[0], G.lg[1]);               // plane passes with one component per CTA
    c->smem_p1 = smem_fast_plane(G.lg[0], G.lg[1], 1);
    c->fb_lgC = fast_mid_lgC(G.lg[2], G.lg[3]);
    if (c->fb_lgC > G.lg[0]) c->fast_b = false;          // the x0 extent must hold one chunk
    c->smem_fa = c->smem_fc = smem_fast_plane(G.lg[0], G.lg[1], 4);
    c->smem_fb = smem_fast_mid(G.lg[2], G.lg[3], c->fb_lgC);
    if (c->fast_a) {
#define X(A, B) if (G.lg[0] == A && G.lg[1] == B) { \
            CK(set_smem(k_fa_delta_fwd<A, B, 6, FAD_NT>, c->smem_fa)); CK(set_smem(k_fa_delta_fwd<A, B, 9, FAD_NT>, c->smem_fa)); \
            CK(set_smem(k_fa_inv<A, B, 4, FC_NT, false>, c->smem_fc)); CK(set_smem(k_fa_inv<A, B, 4, FC_NT, true>, c->smem_fc)); }
        LGF_FAST_PAIRS(X)
#undef X
    }
    if (c->fast_b) {
#define X(A, B) if (G.lg[2] == A && G.lg[3] == B) { \
            CK(set_smem(k_fr_mid<A, B, fast_mid_lgC(A, B), LGF_FR_NT, false>, c->smem_fb)); \
            CK(set_smem(k_fr_mid<A, B, fast_mid_lgC(A, B), LGF_FR_NT, true>, c->smem_fb)); }
        LGF_FAST_PAIRS(X)
#undef X
#define X(A, B) if (G.lg[2] == A && G.lg[3] == B) CK(set_smem(k_fa_mid<A, B, fast_mid_lgC(A, B), fast_mid_nt(A, B)>, c->smem_fb));
        LGF_BIG_PAIRS(X)
#undef X
    }
    c->tma_b = false;
    if (c->fast_b && make_field_tensor_map(c, c->fb_lgC, &c->tm_field)) {
        c->tma_b = true;
#define X(A, B) if (G.lg[2] == A && G.lg[3] == B) \
            c->tma_b = set_smem(k_tb_mid<A, B, fast_mid_lgC(A, B), LGF_TB_NT>, TmaMidGeom<A, B, fast_mid_lgC(A, B)>::SMEM) == cudaSuccess;
        LGF_FAST_PAIRS(X)
#undef X
#define X(A, B) if (G.lg[2] == A && G.lg[3] == B) \
            c->tma_b = set_smem(k_tm_mid<A, B, fast_mid_lgC(A, B), TM1_NT>, TmaBigGeom<A, B, fast_mid_lgC(A, B)>::SMEM) == cudaSuccess;
        LGF_BIG_PAIRS(X)
#undef X
        if (!c->tma_b) cudaGetLastError();
        // the ring form of the 64-extent pass (k_tr_mid): tiles of half the chunk
        c->ring_b = false;
        // (from 2-site chunks on: with 1-site chunks -- 64 x 64 -- the TMA box rows are 16 bytes and the ring measured
        // slower than k_tm_mid, 1065 against 999 us at 64^4)
        if (c->tma_b && big_pair(G.lg[2], G.lg[3]) && c->fb_lgC >= 2 && make_field_tensor_map(c, c->fb_lgC - 1, &c->tm_field_half)) {
#define X(A, B) if (G.lg[2] == A && G.lg[3] == B) \
                c->ring_b = set_smem(k_tr_mid<A, B, fast_mid_lgC(A, B) - 1, TM_NT>, TmaRingGeom<A, B, fast_mid_lgC(A, B) - 1>::SMEM) == cudaSuccess;
            LGF_RING_PAIRS(X)
#undef X
            if (!c->ring_b) cudaGetLastError();
        }
    }
    c->tma_a = false;
#ifndef LGF_F32
    if (c->fast_a && c->NC == 6 && make_link_tensor_maps(c)) {       // 18-real links: two stages do not fit one SM
#define X(A, B) if (G.lg[0] == A && G.lg[1] == B) c->tma_a = set_smem(k_ta_delta_fwd<A, B, 6, 256>, TmaPlaneGeom<A, B, 6>::SMEM) == cudaSuccess;
        LGF_FAST_PAIRS(X)
#undef X
        if (!c->tma_a) cudaGetLastError();
    }
#endif
    c->cl_ok = false;
    if (c->big_p && G.lg[0] == 6 && G.lg[1] == 6) {
        c->smem_cl = smem_fast_plane(6, 6, 2);
        c->cl_ok = set_smem(k_cl_delta_fwd<6, 6, 6, CL_NT>, c->smem_cl) == cudaSuccess &&
                   set_smem(k_cl_delta_fwd<6, 6, 9, CL_NT>, c->smem_cl) == cudaSuccess;
        if (!c->cl_ok) cudaGetLastError();
    }
    if (c->big_p) {
#define X(A, B) if (G.lg[0] == A && G.lg[1] == B) { \
            CK(set_smem(k_fa_fwd<A, B, 1, FC_NT>, c->smem_p1)); CK(set_smem(k_fa_inv<A, B, 1, FC_NT, false>, c->smem_p1)); }
        LGF_BIG_PAIRS(X)
#undef X
    }
    return LGF_OK;
}

lgf_status setup_kernels(lgf_ctx* c) {
    const Geom& G = c->G;
    const int nP = G.L[0] * G.L[1];
    auto smem01 = [&](int ncomp) { return (size_t)((G.L[0] + 1) * G.L[1] * ncomp + G.L[0] + G.L[1]) * sizeof(cplx); };
    c->fft01_ncomp_fused_ok = smem01(4) <= (size_t)MAX_SMEM;
    c->smem01_fused = smem01(4);
    int ncomp = 4;
    while (ncomp > 1 && smem01(ncomp) > 100 * 1024) ncomp >>= 1;
    c->fft01_ncomp = ncomp;
    c->smem01 = smem01(ncomp);
    int th = nP * 4 / 8; if (th > 256) th = 256; if (th < 32) th = 32;
    c->fft01_threads = th;
    // axes 2,3: chunk of x0
    const int n23 = G.L[2] * G.L[3];
    int lgC = 3; if (lgC > G.lg[0]) lgC = G.lg[0];
    while (lgC > 1 && ((size_t)n23 << lgC) * 16 > 64 * 1024) lgC--;
    if (((size_t)n23 << lgC) * 16 > (size_t)MAX_SMEM - 8192) lgC = 0;
    c->fft23_lgC = lgC;
    const int C0 = 1 << lgC;
    c->fft23_S1 = C0;
    c->fft23_S2 = C0 * G.L[2] + (C0 < 8 ? C0 : 0);
    c->smem23 = (size_t)(c->fft23_S2 * G.L[3] + G.L[2] + G.L[3]) * sizeof(cplx) + (size_t)(G.L[2] + G.L[3]) * 8;
    if (c->smem23 > (size_t)MAX_SMEM || c->smem01 > (size_t)MAX_SMEM) return LGF_ERR_UNSUPPORTED;
    th = (n23 << lgC) / 8; if (th > 256) th = 256; if (th < 32) th = 32;
    c->fft23_threads = th;

    CK(set_smem(k_fft01<MODE_FWD, 6>, c->smem01));
    CK(set_smem(k_fft01<MODE_INV, 6>, c->smem01));
    CK(set_smem(k_fft23_mid, c->smem23));
    if (c->fft01_ncomp_fused_ok) {
        CK(set_smem(k_fft01<MODE_DELTA_FWD, 6>, c->smem01_fused));
        CK(set_smem(k_fft01<MODE_DELTA_FWD, 9>, c->smem01_fused));
        CK(set_smem(k_fft01<MODE_INV_G, 6>, c->smem01_fused));
    }
    return setup_fast(c);
}

lgf_status build_tables(lgf_ctx* c) {
    std::vector<real> tw(4 * 128 * 2, real(0));
    std::vector<double> s(4 * 128, 0.0);
    for (int mu = 0; mu < 4; mu++) c->T.plan[mu] = make_plan(c->G.lg[mu], (mu & 1) != 0, mu >= 2);
    const long double pi = 3.141592653589793238462643383279502884L;
    for (int mu = 0; mu < 4; mu++) {
        const int L = c->G.L[mu];
        for (int k = 0; k < L; k++) {
            long double a = 2.0L * pi * (long double)k / (long double)L;
            double cr = (double)cosl(a), sr = (double)sinl(a);
            if ((4 * k) % L == 0) { const int q = 4 * k / L; const double cc[4] = {1, 0, -1, 0}, ss[4] = {0, 1, 0, -1}; cr = cc[q]; sr = ss[q]; }
            tw[(mu * 128 + k) * 2] = (real)cr; tw[(mu * 128 + k) * 2 + 1] = (real)(-sr);
        }
        for (int p = 0; p < L; p++) {
            const int n = stored_freq(p, c->G.lg[mu], c->T.plan[mu]);
            long double sn = sinl(pi * (long double)n / (long double)L);
            s[mu * 128 + p] = (n == 0 || mu >= c->G.nd) ? 0.0 : (double)(4.0L * sn * sn);      // Coulomb: p2 over mu = 0..2
        }
    }
    char* tb = c->ws + c->lay.tables;
    CK(cudaMemcpyAsync(tb, tw.data(), tw.size() * sizeof(real), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(tb + 4 * 128 * 16, s.data(), s.size() * 8, cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    for (int mu = 0; mu < 4; mu++) {
        c->T.tw[mu] = reinterpret_cast<const cplx*>(tb) + mu * 128;
        c->T.s[mu] = reinterpret_cast<const double*>(tb + 4 * 128 * 16) + mu * 128;
    }
    return LGF_OK;
}

// ---- generic kernel launchers -------------------------------------------------------------------------------
template <int NC> void launch_delta(lgf_ctx* c) {
    LaunchScope ls(c, K_DELTA);
    launch_k(c, k_delta<NC>, (unsigned)(c->G.V / 128), 128, 0, c->links, c->field, c->partials, c->G, c->ctl);
}
template <int MODE, int NC> void launch_fft01(lgf_ctx* c, int slot, double half_alpha) {
    LaunchScope ls(c, slot);
    const bool fused = (MODE == MODE_DELTA_FWD || MODE == MODE_INV_G);
    const int ncomp = fused ? 4 : c->fft01_ncomp;
    const unsigned grid = (unsigned)(c->G.L[2] * c->G.L[3] * (4 / ncomp));
    launch_k(c, k_fft01<MODE, NC>, grid, c->fft01_threads, fused ? c->smem01_fused : c->smem01,
        c->field, c->links, c->gbuf, c->partials, c->G, c->T, ncomp, half_alpha, c->ctl);
}
void launch_fft23(lgf_ctx* c) {
    LaunchScope ls(c, K_FFT23_MID);
    const unsigned grid = (unsigned)(4 * c->G.L[1] * (c->G.L[0] >> c->fft23_lgC));
    launch_k(c, k_fft23_mid, grid, c->fft23_threads, c->smem23, c->field, c->G, c->T, c->fft23_lgC, c->fft23_S1, c->fft23_S2,
                                                                   4.0 * (double)c->G.nd / (double)c->G.V, c->ctl);
}
void launch_finalize(lgf_ctx* c, int n_partials) {
    LaunchScope ls(c, K_FINALIZE);
    launch_k(c, k_finalize, 1, n_partials > 8192 ? 1024 : 256, 0, c->partials, n_partials, c->ctl, c->hist, 1.0 / (3.0 * (double)c->G.V), 1.0 / (3.0 * (double)c->G.nd * (double)c->G.V));
}
// S3+S4, g rebuilt from X: one thread per link
// rows walked in bands of 8 values of x2 (k_update_quad<..., LGB = 3>) when a CTA is one x0 row and a time slice of
// links + X outgrows the L2 share
bool update_banded(const lgf_ctx* c) {
    const Geom& G = c->G;
    if (G.L[0] < 64 || G.L[2] < 16) return false;
    const double slice_mb = (double)G.L[0] * G.L[1] * G.L[2] * (2.0 * 4 * c->NC + 4) * sizeof(cplx) / 1e6;
    return slice_mb > 48.0;
}
template <int NC> void launch_update_quad(lgf_ctx* c, double half_alpha) {
    LaunchScope ls(c, K_UPDATE_QUAD);
    cplx* const no_acc = nullptr;
    const bool banded = update_banded(c);
#ifdef LGF_F32
    if (c->acc_g) {                                      // the fp32 phase of LGF_MIXED accumulates the transformation
        if (c->G.L[0] <= 32) launch_k(c, k_update_quad<NC, 32, 1>, (unsigned)(c->G.V / 32), 128, 0, c->links, c->field, c->G, half_alpha, c->ctl, c->gbuf);
        else if (c->G.L[0] == 64) launch_k(c, k_update_quad<NC, 64, 1>, (unsigned)(c->G.V / 64), 256, 0, c->links, c->field, c->G, half_alpha, c->ctl, c->gbuf);
        else launch_k(c, k_update_quad<NC, 128, 1>, (unsigned)(c->G.V / 128), 512, 0, c->links, c->field, c->G, half_alpha, c->ctl, c->gbuf);
        return;
    }
#endif
    if (c->G.L[0] <= 32) launch_k(c, k_update_quad<NC, 32>, (unsigned)(c->G.V / 32), 128, 0, c->links, c->field, c->G, half_alpha, c->ctl, no_acc);
    else if (c->G.L[0] == 64 && banded) launch_k(c, k_update_quad<NC, 64, 0, 3>, (unsigned)(c->G.V / 64), 256, 0, c->links, c->field, c->G, half_alpha, c->ctl, no_acc);
    else if (c->G.L[0] == 64) launch_k(c, k_update_quad<NC, 64>, (unsigned)(c->G.V / 64), 256, 0, c->links, c->field, c->G, half_alpha, c->ctl, no_acc);
    else launch_k(c, k_update_quad<NC, 128>, (unsigned)(c->G.V / 128), 512, 0, c->links, c->field, c->G, half_alpha, c->ctl, no_acc);
}
// S3+S4 with g read from gbuf (LGF_OPT_STORE_G)
template <int NC> void launch_update_g(lgf_ctx* c) {
    LaunchScope ls(c, K_UPDATE_G);
    launch_k(c, k_update_g<NC>, (unsigned)(c->G.V / 128), 128, 0, c->links, c->gbuf, c->G, c->ctl);
}

// ---- kernel selection ------------------------------------------------------------------------------------------
// S1 is fused into pass A wherever the four component tiles of a plane fit one SM (or a CTA pair at 64 x 64)
bool use_fused(const lgf_ctx* c) { return c->fft01_ncomp_fused_ok; }
// the accumulating update of the mixed-precision fp32 phase is k_update_quad only
bool use_store_g(const lgf_ctx* c) { return c->opt_store_g && c->fft01_ncomp_fused_ok && !c->acc_g; }
bool use_fast_a(const lgf_ctx* c) { return c->opt_fast && c->fast_a; }
bool use_fast_b(const lgf_ctx* c) { return c->opt_fast && c->fast_b; }
// pass A with TMA-staged links (Landau gauge; the Coulomb S1 keeps the plain-load kernel)
// -- from two planes per SM on: the persistent grid has one CTA per SM, and below that its tail costs more than the staging
// gains (16^4, 256 planes on 148 SMs: 12.7 against 10.7 us)
// (fp64 only: in the fp32 build the plain-load pass A with its next-site L2 prefetch measured faster, 61.8 against 66.0 us)
bool use_tma_a(const lgf_ctx* c) {
    return sizeof(real) == 8 && c->NC == 6 && c->opt_fast && c->fast_a && c->opt_tma && c->tma_a && c->G.nd == 4 && c->G.L[2] * c->G.L[3] >= 2 * c->sms;
}
bool use_fast_c(const lgf_ctx* c) { return c->opt_fast && c->fast_c; }
bool use_big_p(const lgf_ctx* c) { return c->opt_fast && c->big_p; }
bool use_cluster_a(const lgf_ctx* c) { return use_big_p(c) && c->cl_ok; }
bool use_line_b(const lgf_ctx* c) { return use_fast_b(c) && fast_pair(c->G.lg[2], c->G.lg[3]); }
// ... on TMA-staged tiles (Landau gauge: the Coulomb pass B has no axis-3 phase and keeps the plain-load kernel)
bool use_tma_b(const lgf_ctx* c) { return use_line_b(c) && c->opt_tma && c->tma_b && c->G.nd == 4; }
// 64 extents: the stage-wise pass B with the tile going in and out through the TMA unit (either gauge)
bool use_tma_big(const lgf_ctx* c) { return use_fast_b(c) && !use_line_b(c) && c->opt_tma && c->tma_b; }
// S5 inside pass B's first CTA, where pass B is one of the compile-time-sized kernels
bool use_fin_b(const lgf_ctx* c) { return c->opt_accel && use_fast_b(c); }

// S1 (+ pass A) and, unless pass B does it, the reduction.
template <int NC> void enqueue_head(lgf_ctx* c) {
    int np;
    if (use_tma_a(c)) { launch_ta_delta_fwd(c); np = c->G.L[2] * c->G.L[3]; }
    else if (use_fast_a(c)) { launch_fa_delta_fwd<NC>(c); np = c->G.L[2] * c->G.L[3]; }
    else if (use_cluster_a(c)) { launch_cl_delta_fwd<NC>(c); np = 2 * c->G.L[2] * c->G.L[3]; }
    else if (use_big_p(c)) { launch_delta<NC>(c); np = (int)(c->G.V / 128); launch_fa_fwd1(c); }
    else if (use_fused(c)) { launch_fft01<MODE_DELTA_FWD, NC>(c, K_FFT01_DELTA_FWD, 0.0); np = c->G.L[2] * c->G.L[3]; }
    else { launch_delta<NC>(c); np = (int)(c->G.V / 128); launch_fft01<MODE_FWD, 6>(c, K_FFT01_FWD, 0.0); }
    if (use_fin_b(c)) { c->pending_np = np; return; }     // pass B's CTA 0 reduces them (every head here is followed by a pass B)
    launch_finalize(c, np);
}
void launch_mid(lgf_ctx* c) {
    if (use_tma_b(c)) launch_tb_mid(c); else if (use_tma_big(c) && c->ring_b) launch_tr_mid(c); else if (use_tma_big(c)) launch_tm_mid(c); else if (use_line_b(c)) launch_fr_mid(c); else if (use_fast_b(c)) launch_fa_mid(c); else launch_fft23(c);
}
void launch_inv_x(lgf_ctx* c) {
    if (use_fast_c(c)) launch_fa_inv(c); else if (use_big_p(c)) launch_fa_inv1(c);
    else launch_fft01<MODE_INV, 6>(c, K_FFT01_INV, 0.0);
}
// pass C ending in g (rows 0,1 -> gbuf)
void launch_inv_g(lgf_ctx* c, double half_alpha) {
    if (use_fast_c(c)) launch_fa_inv_g(c, half_alpha); else launch_fft01<MODE_INV_G, 6>(c, K_FFT01_INV_G, half_alpha);
}
template <int NC> void enqueue_tail(lgf_ctx* c, double half_alpha) {
    launch_mid(c);
    if (use_store_g(c)) { launch_inv_g(c, half_alpha); launch_update_g<NC>(c); }
    else { launch_inv_x(c); launch_update_quad<NC>(c, half_alpha); }
}
void enqueue_body(lgf_ctx* c, double half_alpha) {
    if (!c->opt_accel) {
        // plain steepest descent (no Fourier acceleration, PAPER.md:41 refs [1],[2]): X = Delta, so S2 drops out
        if (c->NC == 6) { launch_delta<6>(c); launch_finalize(c, (int)(c->G.V / 128)); launch_update_quad<6>(c, half_alpha); }
        else { launch_delta<9>(c); launch_finalize(c, (int)(c->G.V / 128)); launch_update_quad<9>(c, half_alpha); }
        return;
    }
    if (c->NC == 6) { enqueue_head<6>(c); enqueue_tail<6>(c, half_alpha); }
    else { enqueue_head<9>(c); enqueue_tail<9>(c, half_alpha); }
}
int launches_per_body(const lgf_ctx* c) {
    if (!c->opt_accel) return 3;
    int n;                                               // with a k_finalize launch
    if (use_fast_a(c) || use_cluster_a(c)) n = 5;
    else if (use_big_p(c)) n = 6;
    else n = use_fused(c) ? 5 : 6;
    if (use_fin_b(c)) n -= 1;                            // S5 inside pass B's first CTA
    return n;
}

lgf_status reset_ctl(lgf_ctx* c, double tol, int max_iter) {
    Ctl h; memset(&h, 0, sizeof h);
    h.theta_tol = tol; h.max_iter = max_iter; h.hist_cap = HIST_CAP; h.stall_window = c->stall_window;
    *c->h_ctl = h;
    CK(cudaMemcpyAsync(c->ctl, c->h_ctl, sizeof(Ctl), cudaMemcpyHostToDevice, c->stream));
    return LGF_OK;
}
lgf_status read_ctl(lgf_ctx* c) {
    CK(cudaMemcpyAsync(c->h_ctl, c->ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return LGF_OK;
}

// Enqueue `nb` iteration bodies: a replay of the cached CUDA graph of opt_batch bodies when nb matches, else plain launches.
lgf_status enqueue_bodies(lgf_ctx* c, int nb, double half_alpha) {
    // the legacy default stream cannot be captured: plain launches there
    const bool graph_ok = c->opt_graph && !c->profiling && nb == c->opt_batch && c->stream != nullptr && c->stream != cudaStreamLegacy;
    if (!graph_ok) {
        for (int i = 0; i < nb; i++) enqueue_body(c, half_alpha);
        CK(cudaGetLastError());
        return LGF_OK;
    }
    // Everything that is baked into the captured launches (alpha as a kernel argument, the kernel selection) is kept
    // as a full tuple beside the executable graph and compared member by member: a hash could collide and silently
    // replay a stale graph.
    lgf_ctx::GraphKey key;
    memset(&key, 0, sizeof key);
    key.half_alpha = half_alpha; key.nb = nb; key.nd = c->G.nd; key.acc_g = c->acc_g; key.store_g = use_store_g(c) ? 1 : 0;
    key.fast = c->opt_fast; key.pdl = c->opt_pdl; key.accel = c->opt_accel; key.tma = c->opt_tma;
    if (!c->graph_exec || memcmp(&c->graph_key, &key, sizeof key) != 0) {
        if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
        cudaGraph_t g = nullptr;
        CK(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        c->capturing = true;   // LaunchScope neither counts nor times captured launches
        for (int i = 0; i < nb; i++) enqueue_body(c, half_alpha);
        c->capturing = false;
        CK(cudaStreamEndCapture(c->stream, &g));   // a failed capture is ended (and reported) here
        cudaError_t ge = cudaGraphInstantiate(&c->graph_exec, g, 0);
        cudaGraphDestroy(g);
        if (ge != cudaSuccess) { c->graph_exec = nullptr; CK(ge); }
        c->graph_key = key;
    }
    CK(cudaGraphLaunch(c->graph_exec, c->stream));
    c->launches += (long long)nb * launches_per_body(c);
    return LGF_OK;
}

// Shared driver of lgf_iterate (tol < 0: never) and lgf_fix.
lgf_status run(lgf_ctx* c, double alpha, double tol, int max_iter, bool poll) {
    lgf_status st = reset_ctl(c, tol, max_iter);
    if (st != LGF_OK) return st;
    const double ha = 0.5 * alpha;
    long long bodies_left = (long long)max_iter + 1;
    while (bodies_left > 0) {
        int nb = (int)(bodies_left < c->opt_batch ? bodies_left : c->opt_batch);
        st = enqueue_bodies(c, nb, ha);
        if (st != LGF_OK) return st;
        bodies_left -= nb;
        if (poll || bodies_left == 0) {
            st = read_ctl(c);
            if (st != LGF_OK) return st;
            if (c->h_ctl->done) break;
        }
    }
    if (c->h_ctl->nonfinite) return LGF_ERR_NUMERIC;
    return LGF_OK;
}

// detail of the last failed lgf_create* of this thread (the context it belonged to is gone): lgf_last_error(NULL)
thread_local std::string g_create_err;     // text of this thread's last failed create ("" after a successful one)
#ifndef LGF_F32
thread_local int g_create_from32 = 0;      // 1: that create ran (and failed) in the fp32 translation unit, which keeps its own text
#endif

lgf_status create_impl(const int dims[4], lgf_precision p, lgf_storage s, void* wsp, size_t ws_bytes, void* stream, bool own, lgf_ctx** out) {
    // lgf_last_error(NULL) speaks of the LAST create of this thread: cleared here, set on every failing return below
    g_create_err.clear();
    auto refuse = [&](lgf_status st, const char* why) { g_create_err = why; return st; };
    if (!dims || !out) return refuse(LGF_ERR_INVALID_ARG, "lgf_create: dims or out is NULL");
    *out = nullptr;
    if (p != LGF_FP64 && p != LGF_FP32 && p != LGF_MIXED) return refuse(LGF_ERR_INVALID_ARG, "lgf_create: precision is not LGF_FP64, LGF_FP32 or LGF_MIXED");
    if (s != LGF_STORE_12 && s != LGF_STORE_18) return refuse(LGF_ERR_INVALID_ARG, "lgf_create: storage is not LGF_STORE_12 or LGF_STORE_18");
    for (int k = 0; k < 4; k++) if (dims[k] < 1) return refuse(LGF_ERR_INVALID_ARG, "lgf_create: an extent is smaller than 1");
    if (p != LGF_THIS_PREC) return refuse(LGF_ERR_UNSUPPORTED, "lgf_create: precision not built into this translation unit");
    int lg[4];
    if (!dims_ok(dims, lg)) return refuse(LGF_ERR_UNSUPPORTED, "lgf_create: extents must be powers of two, 4 <= L <= 128, L0*L1 <= 4096, L2*L3 <= 4096");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return refuse(LGF_ERR_CUDA, "lgf_create: no CUDA device (there is no CPU fallback)"); }

    lgf_ctx* c = new (std::nothrow) lgf_ctx();
    if (!c) return refuse(LGF_ERR_OOM, "lgf_create: host allocation of the context failed");
    c->precision = (int)LGF_THIS_PREC;
    int shv = 0;
    for (int k = 0; k < 4; k++) { c->G.L[k] = dims[k]; c->G.lg[k] = lg[k]; c->G.sh[k] = shv; shv += lg[k]; }
    c->G.V = 1LL << shv;
    c->G.nd = 4;
    c->NC = (s == LGF_STORE_12) ? 6 : 9;
    c->lay = make_layout(dims, c->NC);
    c->own_ws = own; c->own_stream = own;
    c->loaded = false;
    c->opt_store_g = 0; c->opt_graph = 1; c->opt_batch = 8; c->opt_fast = 1; c->opt_pdl = 1; c->opt_accel = 1; c->opt_tma = 1;
    { int dev = 0; c->sms = 148; cudaGetDevice(&dev); cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev); if (c->sms < 1) c->sms = 1; }
    c->shadow = nullptr; c->shadow_ws = nullptr; c->acc_g = 0; c->mixed_n32 = 0; c->mixed_switch = 12; c->pending_np = 0; c->stall_window = 0;
    c->graph_exec = nullptr; memset(&c->graph_key, 0, sizeof c->graph_key); c->profiling = 0; c->launches = 0; c->capturing = false;
    c->ev0 = c->ev1 = nullptr; c->h_ctl = nullptr; c->ws = nullptr; c->stream = nullptr; c->copy_stream = nullptr;
    c->ev_copy[0] = c->ev_copy[1] = c->ev_kern[0] = c->ev_kern[1] = nullptr;
    memset(c->prof_ms, 0, sizeof c->prof_ms); memset(c->prof_n, 0, sizeof c->prof_n);

    auto fail = [&](lgf_status st, const char* why = nullptr) {
        g_create_err = !c->err.empty() ? c->err : std::string(why ? why : "lgf_create: set-up failed");
        lgf_destroy(c);
        return st;
    };
    if (own) {
        if (cudaMalloc(&c->ws, c->lay.total) != cudaSuccess) { cudaGetLastError(); return fail(LGF_ERR_OOM, "lgf_create: cudaMalloc of the workspace failed"); }
        if (cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) != cudaSuccess) return fail(LGF_ERR_CUDA, "lgf_create: cudaStreamCreate failed");
    } else {
        if (!wsp || ((size_t)wsp & 255) || ws_bytes < c->lay.total) return fail(LGF_ERR_INVALID_ARG, "lgf_create_ex: workspace is NULL, not 256-byte aligned, or smaller than lgf_workspace_bytes()");
        c->ws = static_cast<char*>(wsp);
        c->stream = static_cast<cudaStream_t>(stream);
    }
    c->links = reinterpret_cast<cplx*>(c->ws + c->lay.links);
    c->field = reinterpret_cast<cplx*>(c->ws + c->lay.field);
    c->gbuf = reinterpret_cast<cplx*>(c->ws + c->lay.gbuf);
    c->staging = reinterpret_cast<dcplx*>(c->ws + c->lay.staging);
    c->partials = reinterpret_cast<double2*>(c->ws + c->lay.partials);
    c->hist = reinterpret_cast<double2*>(c->ws + c->lay.hist);
    c->ctl = reinterpret_cast<Ctl*>(c->ws + c->lay.ctl);
    if (cudaHostAlloc(&c->h_ctl, sizeof(Ctl), cudaHostAllocDefault) != cudaSuccess) return fail(LGF_ERR_OOM, "lgf_create: cudaHostAlloc of the control block failed");
    if (cudaEventCreate(&c->ev0) != cudaSuccess || cudaEventCreate(&c->ev1) != cudaSuccess) return fail(LGF_ERR_CUDA, "lgf_create: cudaEventCreate failed");
    if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(LGF_ERR_CUDA, "lgf_create: cudaStreamCreate (copy stream) failed");
    for (int k = 0; k < 2; k++)
        if (cudaEventCreateWithFlags(&c->ev_copy[k], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_kern[k], cudaEventDisableTiming) != cudaSuccess) return fail(LGF_ERR_CUDA, "lgf_create: cudaEventCreate failed");
    lgf_status st = setup_kernels(c);
    if (st != LGF_OK) return fail(st);
    st = build_tables(c);
    if (st != LGF_OK) return fail(st);
    st = reset_ctl(c, -1.0, 0);
    if (st != LGF_OK) return fail(st);
    *out = c;
    return LGF_OK;
}

// Boundary copies.  The canonical array (array of structs, NE = 9 entries per link; the two-row host format: NE = 6) is
// converted to and from the structure-of-arrays store by k_layout_in/out chunk by chunk.  Host arrays go through two
// staging halves in the workspace: the copies run on the context's copy stream, the layout kernels on its main stream,
// chained by events, so the copy of chunk k+1 overlaps the layout kernel of chunk k (load) and the layout kernel of chunk
// k+1 overlaps the copy of chunk k (get).
lgf_status load_from_device_chunks(lgf_ctx* c, const double* src, bool src_is_host, int NE = 9) {
    const long long V = c->G.V;
    const long long S = src_is_host ? (c->lay.stage_sites + 1) / 2 : c->lay.stage_sites;
    const size_t site_bytes = (size_t)4 * NE * 16;
    if (src_is_host) { CK(cudaEventRecord(c->ev_kern[0], c->stream)); CK(cudaStreamWaitEvent(c->copy_stream, c->ev_kern[0], 0)); }
    int k = 0;
    for (long long off = 0; off < V; off += S, k++) {
        const long long n = (V - off < S) ? V - off : S;
        const int b = k & 1;
        const dcplx* aos;
        if (src_is_host) {
            dcplx* half = c->staging + (size_t)b * S * 36;
            if (k >= 2) CK(cudaStreamWaitEvent(c->copy_stream, c->ev_kern[b], 0));      // the layout kernel of chunk k-2 has read this half
            CK(cudaMemcpyAsync(half, src + off * (4 * NE * 2), (size_t)n * site_bytes, cudaMemcpyHostToDevice, c->copy_stream));
            CK(cudaEventRecord(c->ev_copy[b], c->copy_stream));
            CK(cudaStreamWaitEvent(c->stream, c->ev_copy[b], 0));
            aos = half;
        } else aos = reinterpret_cast<const dcplx*>(src) + off * (4 * NE);
        {
            LaunchScope ls(c, K_LAYOUT_IN);
            const unsigned grid = (unsigned)((n * 4 + 255) / 256);
            if (c->NC == 6) k_layout_in<6><<<grid, 256, 0, c->stream>>>(aos, c->links, V, off, n, NE);
            else k_layout_in<9><<<grid, 256, 0, c->stream>>>(aos, c->links, V, off, n, NE);
        }
        CK(cudaGetLastError());
        if (src_is_host) CK(cudaEventRecord(c->ev_kern[b], c->stream));
    }
    CK(cudaStreamSynchronize(c->stream));
    c->loaded = true;
    return LGF_OK;
}

lgf_status get_to_chunks(lgf_ctx* c, double* dst, bool dst_is_host, int NE = 9) {
    const long long V = c->G.V;
    const long long S = dst_is_host ? (c->lay.stage_sites + 1) / 2 : c->lay.stage_sites;
    const size_t site_bytes = (size_t)4 * NE * 16;
    int k = 0;
    for (long long off = 0; off < V; off += S, k++) {
        const long long n = (V - off < S) ? V - off : S;
        const int b = k & 1;
        dcplx* aos = dst_is_host ? c->staging + (size_t)b * S * 36 : reinterpret_cast<dcplx*>(dst) + off * (4 * NE);
        if (dst_is_host && k >= 2) CK(cudaStreamWaitEvent(c->stream, c->ev_copy[b], 0));            // the copy of chunk k-2 has left this half
        {
            LaunchScope ls(c, K_LAYOUT_OUT);
            const unsigned grid = (unsigned)((n * 4 + 255) / 256);
            if (c->NC == 6) k_layout_out<6><<<grid, 256, 0, c->stream>>>(c->links, aos, V, off, n, NE);
            else k_layout_out<9><<<grid, 256, 0, c->stream>>>(c->links, aos, V, off, n, NE);
        }
        CK(cudaGetLastError());
        if (dst_is_host) {
            CK(cudaEventRecord(c->ev_kern[b], c->stream));
            CK(cudaStreamWaitEvent(c->copy_stream, c->ev_kern[b], 0));
            CK(cudaMemcpyAsync(dst + off * (4 * NE * 2), aos, (size_t)n * site_bytes, cudaMemcpyDeviceToHost, c->copy_stream));
            CK(cudaEventRecord(c->ev_copy[b], c->copy_stream));
        }
    }
    if (dst_is_host) CK(cudaStreamSynchronize(c->copy_stream));
    CK(cudaStreamSynchronize(c->stream));
    return LGF_OK;
}

}  // namespace

extern "C" {

size_t lgf_workspace_bytes(const int dims[4], lgf_precision p, lgf_storage s) {
    int lg[4];
#ifndef LGF_F32
    if (p == LGF_FP32) return lgf32_workspace_bytes(dims, p, s);
    if (p == LGF_MIXED) {
        const size_t n64 = lgf_workspace_bytes(dims, LGF_FP64, s), n32 = lgf32_workspace_bytes(dims, LGF_FP32, s);
        return (n64 && n32) ? align_up(n64, 256) + n32 : 0;
    }
#endif
    if (!dims || p != LGF_THIS_PREC || (s != LGF_STORE_12 && s != LGF_STORE_18) || !dims_ok(dims, lg)) return 0;
    return make_layout(dims, s == LGF_STORE_12 ? 6 : 9).total;
}

#ifndef LGF_F32
// LGF_MIXED: an fp64 context that owns an fp32 shadow context on the same stream
static lgf_status create_mixed(const int dims[4], lgf_storage s, void* ws, size_t bytes, void* stream, bool own, lgf_ctx** out) {
    g_create_err.clear();
    if (!dims || !out) { g_create_err = "lgf_create: dims or out is NULL"; return LGF_ERR_INVALID_ARG; }
    *out = nullptr;
    const size_t n64 = lgf_workspace_bytes(dims, LGF_FP64, s), n32 = lgf32_workspace_bytes(dims, LGF_FP32, s);
    lgf_ctx* c = nullptr;
    lgf_status st;
    if (own) st = create_impl(dims, LGF_FP64, s, nullptr, 0, nullptr, true, &c);
    else {
        if (n64 == 0 || n32 == 0) return create_impl(dims, LGF_FP64, s, ws, bytes, stream, false, &c);   // reports the argument error
        if (!ws || bytes < align_up(n64, 256) + n32) { g_create_err = "lgf_create_ex: LGF_MIXED workspace is NULL or smaller than lgf_workspace_bytes()"; return LGF_ERR_INVALID_ARG; }
        st = create_impl(dims, LGF_FP64, s, ws, align_up(n64, 256), stream, false, &c);
    }
    if (st != LGF_OK) return st;
    char* ws32;
    if (own) {
        if (cudaMalloc(&c->shadow_ws, n32) != cudaSuccess) { cudaGetLastError(); lgf_destroy(c); g_create_err = "lgf_create: cudaMalloc of the fp32 workspace of LGF_MIXED failed"; return LGF_ERR_OOM; }
        ws32 = c->shadow_ws;
    } else ws32 = static_cast<char*>(ws) + align_up(n64, 256);
    st = lgf32_create_ex(dims, LGF_FP32, s, ws32, n32, c->stream, &c->shadow);
    if (st != LGF_OK) { c->shadow = nullptr; lgf_destroy(c); g_create_from32 = 1; return st; }   // the text is the fp32 unit's
    *out = c;
    return LGF_OK;
}
#endif

lgf_status lgf_create(const int dims[4], lgf_precision p, lgf_storage s, lgf_ctx** out) {
#ifndef LGF_F32
    g_create_from32 = (p == LGF_FP32);
    if (p == LGF_FP32) return lgf32_create(dims, p, s, out);
    if (p == LGF_MIXED) return create_mixed(dims, s, nullptr, 0, nullptr, true, out);
#endif
    return create_impl(dims, p, s, nullptr, 0, nullptr, true, out);
}
lgf_status lgf_create_ex(const int dims[4], lgf_precision p, lgf_storage s, void* ws, size_t bytes, void* stream, lgf_ctx** out) {
#ifndef LGF_F32
    g_create_from32 = (p == LGF_FP32);
    if (p == LGF_FP32) return lgf32_create_ex(dims, p, s, ws, bytes, stream, out);
    if (p == LGF_MIXED) return create_mixed(dims, s, ws, bytes, stream, false, out);
#endif
    return create_impl(dims, p, s, ws, bytes, stream, false, out);
}

void lgf_destroy(lgf_ctx* c) {
    FWD32V(lgf32_destroy(c))
    if (!c) return;
    if (c->stream) cudaStreamSynchronize(c->stream);
#ifndef LGF_F32
    if (c->shadow) lgf32_destroy(c->shadow);
    if (c->shadow_ws) cudaFree(c->shadow_ws);
#endif
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    for (int k = 0; k < 2; k++) { if (c->ev_copy[k]) cudaEventDestroy(c->ev_copy[k]); if (c->ev_kern[k]) cudaEventDestroy(c->ev_kern[k]); }
    if (c->copy_stream) { cudaStreamSynchronize(c->copy_stream); cudaStreamDestroy(c->copy_stream); }
    if (c->h_ctl) cudaFreeHost(c->h_ctl);
    if (c->own_ws && c->ws) cudaFree(c->ws);
    if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
    delete c;
}

lgf_status lgf_load_links(lgf_ctx* c, const double* host_links) {
    FWD32(lgf32_load_links(c, host_links))
    if (!c || !host_links) return LGF_ERR_INVALID_ARG;
    return load_from_device_chunks(c, host_links, true);
}
lgf_status lgf_load_links_device(lgf_ctx* c, const double* dev_links) {
    FWD32(lgf32_load_links_device(c, dev_links))
    if (!c || !dev_links) return LGF_ERR_INVALID_ARG;
    return load_from_device_chunks(c, dev_links, false);
}
lgf_status lgf_load_links_12(lgf_ctx* c, const double* host_rows) {
    FWD32(lgf32_load_links_12(c, host_rows))
    if (!c || !host_rows) return LGF_ERR_INVALID_ARG;
    if (c->NC != 6) return LGF_ERR_UNSUPPORTED;          // the two-row host format goes with two-row storage
    return load_from_device_chunks(c, host_rows, true, 6);
}
lgf_status lgf_get_links_12(lgf_ctx* c, double* host_rows) {
    FWD32(lgf32_get_links_12(c, host_rows))
    if (!c || !host_rows) return LGF_ERR_INVALID_ARG;
    if (c->NC != 6) return LGF_ERR_UNSUPPORTED;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    return get_to_chunks(c, host_rows, true, 6);
}
lgf_status lgf_get_links(lgf_ctx* c, double* host_links) {
    FWD32(lgf32_get_links(c, host_links))
    if (!c || !host_links) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    return get_to_chunks(c, host_links, true);
}
lgf_status lgf_get_links_device(lgf_ctx* c, double* dev_links) {
    FWD32(lgf32_get_links_device(c, dev_links))
    if (!c || !dev_links) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    return get_to_chunks(c, dev_links, false);
}

#ifdef LGF_F32
void* lgf32_x_begin(lgf_ctx* c) {
    c->loaded = true; c->acc_g = 1;
    c->stall_window = LGF_MIXED_STALL_WINDOW;
    LaunchScope ls(c, K_MISC);
    k_init_gacc<<<(unsigned)((c->G.V + 255) / 256), 256, 0, c->stream>>>(c->gbuf, c->G.V);
    return c->links;
}
void* lgf32_x_gacc(lgf_ctx* c) { return c->gbuf; }
#endif

lgf_status lgf_iterate(lgf_ctx* c, int n, double alpha, double* F, double* theta) {
    FWD32(lgf32_iterate(c, n, alpha, F, theta))
    if (!c || n < 0 || !(alpha > 0.0) || !std::isfinite(alpha)) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    lgf_status st = run(c, alpha, -1.0, n, false);
    if (st != LGF_OK) return st;
    if (F) *F = c->h_ctl->F;
    if (theta) *theta = c->h_ctl->theta;
    return LGF_OK;
}

lgf_status lgf_fix(lgf_ctx* c, double alpha, double theta_tol, int max_iter, int* n_iter, double* F, double* theta) {
    FWD32(lgf32_fix(c, alpha, theta_tol, max_iter, n_iter, F, theta))
    if (!c || max_iter < 0 || !(alpha > 0.0) || !std::isfinite(alpha) || !(theta_tol >= 0.0)) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    int n32 = 0;
#ifndef LGF_F32
    if (c->shadow) {
        // Mixed precision.  Phase 1: a float copy of the links is fixed in fp32 down to theta_sw while the fp32 update
        // accumulates the total transformation Gacc(x).  The fp32 floor of theta is 1e-14..1e-12 (round-off of Delta
        // amplified by p2max/p2min, which grows as L^2), so theta_sw may be out of reach: the phase also ends when theta
        // has not halved within LGF_MIXED_STALL_WINDOW iterations (stagnation guard, Ctl::stall_window) -- never by
        // exhausting max_iter on a stalled fp32 run.  Phase 2: the fp64 links receive Gacc in one step (re-orthonormalised
        // in double: an exact gauge copy of the input) and the fp64 iteration takes theta to theta_tol with the remaining
        // budget.
        const double sw = pow(10.0, -(double)c->mixed_switch);
        const double theta_sw = theta_tol > sw ? theta_tol : sw;
        float2* l32 = static_cast<float2*>(lgf32_x_begin(c->shadow));
        const long long n = 4LL * c->NC * c->G.V;
        { LaunchScope ls(c, K_MISC); k_demote<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->links, l32, n); }
        CK(cudaGetLastError());
        double F32v = 0, th32 = 0;
        lgf_status s1 = lgf32_fix(c->shadow, alpha, theta_sw, max_iter, &n32, &F32v, &th32);
        if (s1 != LGF_OK && s1 != LGF_NOT_CONVERGED) { c->err = std::string("fp32 phase: ") + lgf32_last_error(c->shadow); return s1; }
        {
            LaunchScope ls(c, K_MISC);
            const float2* ga = static_cast<const float2*>(lgf32_x_gacc(c->shadow));
            if (c->NC == 6) k_apply_gacc<6><<<(unsigned)(4 * (c->G.V / 128)), 128, 0, c->stream>>>(c->links, ga, c->G);
            else k_apply_gacc<9><<<(unsigned)(4 * (c->G.V / 128)), 128, 0, c->stream>>>(c->links, ga, c->G);
        }
        CK(cudaGetLastError());
        c->mixed_n32 = n32;
        max_iter = max_iter > n32 ? max_iter - n32 : 0;
    }
#endif
    lgf_status st = run(c, alpha, theta_tol, max_iter, true);
    if (st != LGF_OK) return st;
    if (n_iter) *n_iter = n32 + c->h_ctl->iters;
    if (F) *F = c->h_ctl->F;
    if (theta) *theta = c->h_ctl->theta;
    return c->h_ctl->converged ? LGF_OK : LGF_NOT_CONVERGED;
}

// Step-size scan (PAPER.md:47 fixes one alpha = 0.08, its refs [1],[2] tune it): the same start,
// one lgf_fix per alpha, the iteration counts side by side.  The start is kept in a temporary device copy of the link
// store and put back at the end, so the context's links are unchanged by the call.
lgf_status lgf_scan_alpha(lgf_ctx* c, const double* alphas, int n, double theta_tol, int max_iter, int* counts, double* F_final, int* best) {
    FWD32(lgf32_scan_alpha(c, alphas, n, theta_tol, max_iter, counts, F_final, best))
    if (!c || !alphas || !counts || n < 1 || max_iter < 0 || !(theta_tol >= 0.0)) return LGF_ERR_INVALID_ARG;
    for (int k = 0; k < n; k++) if (!(alphas[k] > 0.0) || !std::isfinite(alphas[k])) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    const size_t bytes = (size_t)c->G.V * 4 * c->NC * sizeof(cplx);
    void* keep = nullptr;
    if (cudaMalloc(&keep, bytes) != cudaSuccess) { cudaGetLastError(); return LGF_ERR_OOM; }
    lgf_status out = LGF_OK;
    auto copy = [&](void* dst, const void* src) { return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, c->stream) == cudaSuccess; };
    if (!copy(keep, c->links)) out = LGF_ERR_CUDA;
    int arg = -1;
    for (int k = 0; k < n && out == LGF_OK; k++) {
        if (k > 0 && !copy(c->links, keep)) { out = LGF_ERR_CUDA; break; }
        int it = 0; double F = 0, th = 0;
        const lgf_status st = lgf_fix(c, alphas[k], theta_tol, max_iter, &it, &F, &th);
        if (st == LGF_OK) { counts[k] = it; if (arg < 0 || it < counts[arg]) arg = k; }
        else if (st == LGF_NOT_CONVERGED) counts[k] = -1;         // max_iter updates did not reach theta_tol
        else if (st == LGF_ERR_NUMERIC) counts[k] = -2;           // this alpha diverges
        else { out = st; break; }
        if (F_final) F_final[k] = (st == LGF_ERR_NUMERIC) ? 0.0 : F;
    }
    if (!copy(c->links, keep) && out == LGF_OK) out = LGF_ERR_CUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess && out == LGF_OK) out = LGF_ERR_CUDA;
    cudaFree(keep);
    if (out == LGF_OK && best) *best = arg;
    return out;
}

lgf_status lgf_measure(lgf_ctx* c, double* F, double* theta, double* plaq) {
    FWD32(lgf32_measure(c, F, theta, plaq))
    if (!c) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    lgf_status st = reset_ctl(c, -1.0, 0);
    if (st != LGF_OK) return st;
    if (c->NC == 6) launch_delta<6>(c); else launch_delta<9>(c);
    launch_finalize(c, (int)(c->G.V / 128));
    {
        LaunchScope ls(c, K_PLAQUETTE);
        if (c->NC == 6) k_plaquette<6><<<(unsigned)(c->G.V / 128), 128, 0, c->stream>>>(c->links, c->partials, c->G);
        else k_plaquette<9><<<(unsigned)(c->G.V / 128), 128, 0, c->stream>>>(c->links, c->partials, c->G);
    }
    double* sums = reinterpret_cast<double*>(c->ws + c->lay.scratch);
    {
        LaunchScope ls(c, K_MISC);
        k_sum_partials<<<1, 256, 0, c->stream>>>(c->partials, (int)(c->G.V / 128), sums);
    }
    CK(cudaGetLastError());
    double h[2];
    CK(cudaMemcpyAsync(h, sums, 16, cudaMemcpyDeviceToHost, c->stream));
    st = read_ctl(c);
    if (st != LGF_OK) return st;
    if (c->h_ctl->nonfinite) return LGF_ERR_NUMERIC;
    if (F) *F = c->h_ctl->F;
    if (theta) *theta = c->h_ctl->theta;
    if (plaq) *plaq = h[0] / (18.0 * (double)c->G.V);
    return LGF_OK;
}

lgf_status lgf_get_history(lgf_ctx* c, double* hist, int capacity, int* n_out) {
    FWD32(lgf32_get_history(c, hist, capacity, n_out))
    if (!c || !hist || capacity < 0 || !n_out) return LGF_ERR_INVALID_ARG;
    int n = c->h_ctl->n_meas; if (n > HIST_CAP) n = HIST_CAP; if (n > capacity) n = capacity;
    if (n > 0) {
        CK(cudaMemcpyAsync(hist, c->hist, (size_t)n * 16, cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
    }
    *n_out = n;
    return LGF_OK;
}

lgf_status lgf_get_field(lgf_ctx* c, lgf_field which, double alpha, double* host_field) {
    FWD32(lgf32_get_field(c, which, alpha, host_field))
    if (!c || !host_field) return LGF_ERR_INVALID_ARG;
    if (which != LGF_FIELD_DELTA && which != LGF_FIELD_X && which != LGF_FIELD_G) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    lgf_status st = reset_ctl(c, -1.0, 1 << 30);
    if (st != LGF_OK) return st;
    const double ha = 0.5 * alpha;
    bool g_from_buf = false;
    if (which == LGF_FIELD_DELTA || !c->opt_accel) {       // plain steepest descent: X = Delta
        if (c->NC == 6) launch_delta<6>(c); else launch_delta<9>(c);
    } else {
        if (c->NC == 6) enqueue_head<6>(c); else enqueue_head<9>(c);
        launch_mid(c);
        if (which == LGF_FIELD_G && use_store_g(c)) { launch_inv_g(c, ha); g_from_buf = true; }
        else launch_inv_x(c);
    }
    CK(cudaGetLastError());
    const long long V = c->G.V;
    const long long S = c->lay.stage_sites * 4;   // staging holds 4*9 complex per site -> 4x as many 3x3 matrices
    for (long long off = 0; off < V; off += S) {
        const long long n = (V - off < S) ? V - off : S;
        {
            LaunchScope ls(c, K_MISC);
            const unsigned grid = (unsigned)((n + 255) / 256);
            if (which == LGF_FIELD_G) k_unpack_g<<<grid, 256, 0, c->stream>>>(g_from_buf ? c->gbuf : c->field, g_from_buf ? 0 : 1, ha, c->staging, V, off, n);
            else k_unpack_field<<<grid, 256, 0, c->stream>>>(c->field, c->staging, V, off, n);
        }
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(host_field + off * 18, c->staging, (size_t)n * 144, cudaMemcpyDeviceToHost, c->stream));
    }
    CK(cudaStreamSynchronize(c->stream));
    return LGF_OK;
}

lgf_status lgf_set_option(lgf_ctx* c, lgf_option opt, int value) {
    FWD32(lgf32_set_option(c, opt, value))
    if (!c) return LGF_ERR_INVALID_ARG;
#ifndef LGF_F32
    if (c->shadow && (opt == LGF_OPT_GAUGE_DIRECTIONS || opt == LGF_OPT_FOURIER_ACCEL)) {      // the method itself: both phases
        lgf_status st = lgf32_set_option(c->shadow, opt, value);
        if (st != LGF_OK) return st;
    }
#endif
    switch (opt) {
        case LGF_OPT_STORE_G: c->opt_store_g = value ? 1 : 0; break;
        case LGF_OPT_GRAPH: c->opt_graph = value ? 1 : 0; break;
        case LGF_OPT_BATCH: if (value < 1 || value > 1024) return LGF_ERR_INVALID_ARG; c->opt_batch = value; break;
        case LGF_OPT_PDL: c->opt_pdl = value ? 1 : 0; break;
        case LGF_OPT_FAST_FFT: c->opt_fast = value ? 1 : 0; break;
        case LGF_OPT_TMA: c->opt_tma = value ? 1 : 0; break;
        case LGF_OPT_FOURIER_ACCEL: c->opt_accel = value ? 1 : 0; break;
        case LGF_OPT_MIXED_SWITCH: if (value < 4 || value > 20) return LGF_ERR_INVALID_ARG; c->mixed_switch = value; break;
        case LGF_OPT_GAUGE_DIRECTIONS: {
            if (value != 3 && value != 4) return LGF_ERR_INVALID_ARG;
            c->G.nd = value;
            lgf_status st = build_tables(c);         // the p2 table of axis 3 is zero in Coulomb gauge
            if (st != LGF_OK) return st;
            break;
        }
        default: return LGF_ERR_INVALID_ARG;
    }
    return LGF_OK;
}
lgf_status lgf_get_option(lgf_ctx* c, lgf_option opt, int* value) {
    FWD32(lgf32_get_option(c, opt, value))
    if (!c || !value) return LGF_ERR_INVALID_ARG;
    switch (opt) {
        case LGF_OPT_STORE_G: *value = use_store_g(c) ? 1 : 0; break;
        case LGF_OPT_GRAPH: *value = c->opt_graph; break;
        case LGF_OPT_BATCH: *value = c->opt_batch; break;
        case LGF_OPT_PDL: *value = c->opt_pdl; break;
        case LGF_OPT_FAST_FFT: *value = ((use_fast_a(c) || use_big_p(c)) ? 1 : 0) | (use_fast_b(c) ? 2 : 0) | ((use_fast_c(c) || use_big_p(c)) ? 4 : 0); break;
        case LGF_OPT_TMA: *value = ((use_tma_b(c) || use_tma_big(c)) ? 1 : 0) | (use_tma_a(c) ? 2 : 0); break;
        case LGF_OPT_FOURIER_ACCEL: *value = c->opt_accel; break;
        case LGF_OPT_GAUGE_DIRECTIONS: *value = c->G.nd; break;
        case LGF_OPT_MIXED_FP32_ITERS: *value = c->mixed_n32; break;
        case LGF_OPT_MIXED_SWITCH: *value = c->mixed_switch; break;
        default: return LGF_ERR_INVALID_ARG;
    }
    return LGF_OK;
}

lgf_status lgf_set_profiling(lgf_ctx* c, int on) {
    FWD32(lgf32_set_profiling(c, on))
    if (!c) return LGF_ERR_INVALID_ARG;
    prof_flush(c);
    c->profiling = on ? 1 : 0;
    memset(c->prof_ms, 0, sizeof c->prof_ms); memset(c->prof_n, 0, sizeof c->prof_n);
    return LGF_OK;
}
lgf_status lgf_get_profile(lgf_ctx* c, double ms[LGF_MAX_KERNELS], long long n[LGF_MAX_KERNELS]) {
    FWD32(lgf32_get_profile(c, ms, n))
    if (!c || !ms || !n) return LGF_ERR_INVALID_ARG;
    prof_flush(c);
    memcpy(ms, c->prof_ms, sizeof c->prof_ms); memcpy(n, c->prof_n, sizeof c->prof_n);
    return LGF_OK;
}
#ifndef LGF_F32
const char* lgf_kernel_name(int slot) { return (slot >= 0 && slot < K_NSLOTS) ? kKernelNames[slot] : ""; }
#endif
long long lgf_launch_count(lgf_ctx* c) {
    FWD32(lgf32_launch_count(c))
    return c ? c->launches : 0;
}

#ifndef LGF_F32
lgf_status lgf_copy_peak(void* dst, const void* src, size_t bytes, int reps, void* stream, double* ms) {
    if (!dst || !src || !ms || reps < 1 || bytes < 16 || (bytes & 15)) return LGF_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return LGF_ERR_CUDA;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long n = (long long)(bytes / 16);
    const unsigned grid = (unsigned)(sms * 8);
    k_copy<<<grid, 256, 0, s>>>((double2*)dst, (const double2*)src, n);   // warm-up
    cudaEventRecord(a, s);
    for (int i = 0; i < reps; i++) k_copy<<<grid, 256, 0, s>>>((double2*)dst, (const double2*)src, n);
    cudaEventRecord(b, s);
    cudaError_t e = cudaEventSynchronize(b);
    float t = 0; cudaEventElapsedTime(&t, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return LGF_ERR_CUDA;
    *ms = (double)t / reps;
    return LGF_OK;
}

lgf_status lgf_stream_peak(void* buf, size_t n_sites, int write, int reps, void* stream, double* ms) {
    if (!buf || !ms || reps < 1 || n_sites < 128 || (n_sites & 127)) return LGF_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return LGF_ERR_CUDA;
    double2* p = static_cast<double2*>(buf);
    const unsigned grid = (unsigned)(n_sites / 128);
    const long long V = (long long)n_sites;
    for (int i = -1; i < reps; i++) {
        if (i == 0) cudaEventRecord(a, s);
        if (write) k_streams<1><<<grid, 128, 0, s>>>(p, V, p); else k_streams<0><<<grid, 128, 0, s>>>(p, V, p);
    }
    cudaEventRecord(b, s);
    cudaError_t e = cudaEventSynchronize(b);
    float t = 0; cudaEventElapsedTime(&t, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return LGF_ERR_CUDA;
    *ms = (double)t / reps;
    return LGF_OK;
}

lgf_status lgf_fp64_peak(int reps, void* stream, double* tflops) {
    if (!tflops || reps < 1) return LGF_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return LGF_ERR_CUDA;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    double* sink = nullptr;
    if (cudaMalloc(&sink, 8) != cudaSuccess) { cudaGetLastError(); cudaEventDestroy(a); cudaEventDestroy(b); return LGF_ERR_OOM; }
    const int iters = 4096;
    const unsigned grid = (unsigned)(sms * 8);                        // 8 CTAs of 256 threads per SM: 64 warps
    k_fma64<<<grid, 256, 0, s>>>(sink, iters, 0.999999, 1e-9);        // warm-up
    cudaEventRecord(a, s);
    for (int i = 0; i < reps; i++) k_fma64<<<grid, 256, 0, s>>>(sink, iters, 0.999999, 1e-9);
    cudaEventRecord(b, s);
    cudaError_t e = cudaEventSynchronize(b);
    float t = 0; cudaEventElapsedTime(&t, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(sink);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return LGF_ERR_CUDA;
    *tflops = 2.0 * 8.0 * iters * 256.0 * grid * reps / ((double)t * 1e-3) / 1e12;
    return LGF_OK;
}

const char* lgf_status_string(lgf_status s) {
    switch (s) {
        case LGF_OK: return "ok";
        case LGF_ERR_INVALID_ARG: return "invalid argument";
        case LGF_ERR_UNSUPPORTED: return "unsupported lattice size or precision";
        case LGF_ERR_OOM: return "out of memory";
        case LGF_ERR_CUDA: return "CUDA error (or no CUDA device: there is no CPU fallback)";
        case LGF_ERR_NOT_LOADED: return "links not loaded";
        case LGF_ERR_NUMERIC: return "theta or F is not finite";
        case LGF_NOT_CONVERGED: return "max_iter reached before theta < theta_tol";
    }
    return "unknown status";
}
#endif
const char* lgf_last_error(lgf_ctx* c) {
    FWD32(lgf32_last_error(c))
#ifndef LGF_F32
    if (!c && g_create_from32) return lgf32_last_error(nullptr);     // the last create of this thread failed in the fp32 unit
#endif
    return c ? c->err.c_str() : g_create_err.c_str();
}

}  // extern "C"

#ifndef LGF_F32
#include "lgf_slab.inl"
#endif
