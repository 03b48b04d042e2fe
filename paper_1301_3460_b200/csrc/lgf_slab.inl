// lgf_slab.inl -- host side of the slab-decomposed context (include/lgf.h lgf_*_sharded; kernels in slab.cuh).
// Included by lgf_api.cu in the fp64 build only.
//
// P ranks, each with its OWN workspace (its own cudaMalloc), all on the current device and on one stream: "virtual
// ranks".  Everything a rank touches of another rank goes through exactly two doors, and both are written so that the
// ranks can be real GPUs with peer access:
//   slab_copy2d()   the halo exchanges (cudaMemcpy2DAsync between two ranks' workspaces: a device copy here,
//                   a peer copy over NVLink -- or ncclSend/ncclRecv -- between GPUs)
//   SlabPeers       the table of peer pointers k_slab_scatter / k_slab_gather store through (NVLink P2P stores).
// The only other shared state is the (theta, F) reduction and the stop flag: here one partials array and one control
// block on the device; between GPUs an all-reduce of two doubles per iteration, summed in rank order.
#include "slab.cuh"

struct lgf_slab_ctx {
    int P, lgP, NC;
    Geom Gg, Gl, Gt;                     // global lattice, a rank's slab (L0,L1,L2,L3/P), a rank's transposed lattice (L0,L1/P,L2,L3)
    long long Vl, S;                     // sites per rank, sites per time slice
    cudaStream_t stream;
    char* ws[SLAB_MAX_RANKS];            // one workspace per rank
    cplx *links[SLAB_MAX_RANKS], *field[SLAB_MAX_RANKS], *fieldT[SLAB_MAX_RANKS], *halo_u[SLAB_MAX_RANKS], *halo_x[SLAB_MAX_RANKS];
    char* shared;                        // partials of all ranks, control block, history, FFT tables
    double2 *partials, *hist;
    Ctl *ctl, *h_ctl;
    FftTables Tl, Tt[SLAB_MAX_RANKS];    // Tt[r]: the p^2 table of axis 1 starts at rank r's first x1
    int nb;                              // S1 partials per rank
    int fft01_ncomp, fft01_threads, fft23_lgC, fft23_S2, fft23_threads;
    size_t smem01, smem23;
    bool loaded;
    long long launches, copies;
    cudaError_t copy_err;                // first failed inter-rank copy since the last slab_run began (cudaSuccess: none)
    const char* copy_what;
    std::string err;
};

namespace {

thread_local std::string g_slab_create_err;      // text of this thread's last failed lgf_create_sharded ("" after a success)

#define SCK(call)                                                                                          \
    do {                                                                                                   \
        cudaError_t e_ = (call);                                                                           \
        if (e_ != cudaSuccess) {                                                                           \
            char b_[512];                                                                                  \
            snprintf(b_, sizeof b_, "%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            c->err = b_;                                                                                   \
            return LGF_ERR_CUDA;                                                                           \
        }                                                                                                  \
    } while (0)

// THE inter-rank copy: `rows` runs of `row_bytes` each, source and destination pitches in bytes.  Virtual ranks: a
// device-to-device copy.  Real GPUs: cudaMemcpy2DAsync with cudaMemcpyDefault over peer-mapped pointers is the same call
// (the runtime routes it over NVLink), or an ncclSend/ncclRecv pair of the packed rows.
cudaError_t slab_copy2d(void* dst, size_t dpitch, const void* src, size_t spitch, size_t row_bytes, size_t rows, cudaStream_t s) {
    return cudaMemcpy2DAsync(dst, dpitch, src, spitch, row_bytes, rows, cudaMemcpyDefault, s);
}

// The halo exchanges are enqueued from functions that return nothing; a failed copy is remembered here and turned into
// LGF_ERR_CUDA by slab_run before any result is read.
void slab_exchange(lgf_slab_ctx* c, const char* what, void* dst, size_t dpitch, const void* src, size_t spitch, size_t row_bytes, size_t rows) {
    const cudaError_t e = slab_copy2d(dst, dpitch, src, spitch, row_bytes, rows, c->stream);
    if (e != cudaSuccess && c->copy_err == cudaSuccess) { c->copy_err = e; c->copy_what = what; }
    c->copies++;
}

void slab_geom(Geom& G, int l0, int l1, int l2, int l3, int nd) {
    const int lg[4] = {l0, l1, l2, l3};
    int sh = 0;
    for (int k = 0; k < 4; k++) { G.L[k] = 1 << lg[k]; G.lg[k] = lg[k]; G.sh[k] = sh; sh += lg[k]; }
    G.V = 1LL << sh;
    G.nd = nd;
}

lgf_status slab_reset_ctl(lgf_slab_ctx* c, double tol, int max_iter) {
    Ctl h; memset(&h, 0, sizeof h);
    h.theta_tol = tol; h.max_iter = max_iter; h.hist_cap = HIST_CAP;
    *c->h_ctl = h;
    SCK(cudaMemcpyAsync(c->ctl, c->h_ctl, sizeof(Ctl), cudaMemcpyHostToDevice, c->stream));
    return LGF_OK;
}
lgf_status slab_read_ctl(lgf_slab_ctx* c) {
    SCK(cudaMemcpyAsync(c->h_ctl, c->ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, c->stream));
    SCK(cudaStreamSynchronize(c->stream));
    return LGF_OK;
}

// S1 on every rank (after the U_3 halo exchange) and the reduction over all ranks' partials in rank order.
template <int NC> void slab_measure(lgf_slab_ctx* c) {
    const int P = c->P;
    for (int r = 0; r < P; r++) {                        // halo 1: U_3 of the last slice of rank r-1 -> rank r
        const int q = (r + P - 1) % P;
        const cplx* src = c->links[q] + (long long)(3 * NC) * c->Vl + (c->Vl - c->S);
        slab_exchange(c, "U_3 halo", c->halo_u[r], (size_t)c->S * sizeof(cplx), src, (size_t)c->Vl * sizeof(cplx), (size_t)c->S * sizeof(cplx), NC);
    }
    for (int r = 0; r < P; r++) {
        k_delta_slab<NC><<<(unsigned)c->nb, 128, 0, c->stream>>>(c->links[r], c->halo_u[r], c->field[r], c->partials + (size_t)r * c->nb, c->Gl, c->ctl);
        c->launches++;
    }
    const int np = P * c->nb;
    k_finalize<<<1, np > 8192 ? 1024 : 256, 0, c->stream>>>(c->partials, np, c->ctl, c->hist, 1.0 / (3.0 * (double)c->Gg.V), 1.0 / (12.0 * (double)c->Gg.V));
    c->launches++;
}

template <int NC> void slab_body(lgf_slab_ctx* c, double half_alpha) {
    const int P = c->P;
    const Geom& Gl = c->Gl; const Geom& Gt = c->Gt;
    slab_measure<NC>(c);
    cplx* const none = nullptr; double2* const nop = nullptr;
    const unsigned g01 = (unsigned)(Gl.L[2] * Gl.L[3] * (4 / c->fft01_ncomp));
    for (int r = 0; r < P; r++) {                        // pass A, local
        k_fft01<MODE_FWD, 6><<<g01, c->fft01_threads, c->smem01, c->stream>>>(c->field[r], none, none, nop, Gl, c->Tl, c->fft01_ncomp, 0.0, c->ctl);
        c->launches++;
    }
    SlabPeers pt, pf;
    for (int r = 0; r < SLAB_MAX_RANKS; r++) { pt.p[r] = r < P ? c->fieldT[r] : nullptr; pf.p[r] = r < P ? c->field[r] : nullptr; }
    const unsigned gtr = (unsigned)((c->Vl + 255) / 256);
    for (int r = 0; r < P; r++) {                        // transpose: x3 split -> x1 split
        k_slab_scatter<<<gtr, 256, 0, c->stream>>>(c->field[r], pt, r, Gl.lg[0], Gl.lg[1], Gl.lg[2], Gl.lg[3], c->lgP, c->ctl);
        c->launches++;
    }
    const unsigned g23 = (unsigned)(4 * Gt.L[1] * (Gt.L[0] >> c->fft23_lgC));
    const double scale = 16.0 / (double)c->Gg.V;         // p2max / V of the WHOLE lattice
    for (int r = 0; r < P; r++) {                        // pass B, local on the transposed lattice
        k_fft23_mid<<<g23, c->fft23_threads, c->smem23, c->stream>>>(c->fieldT[r], Gt, c->Tt[r], c->fft23_lgC, 1 << c->fft23_lgC, c->fft23_S2, scale, c->ctl);
        c->launches++;
    }
    for (int r = 0; r < P; r++) {                        // transpose back
        k_slab_gather<<<gtr, 256, 0, c->stream>>>(c->fieldT[r], pf, r, Gl.lg[0], Gl.lg[1], Gl.lg[2], Gl.lg[3], c->lgP, c->ctl);
        c->launches++;
    }
    for (int r = 0; r < P; r++) {                        // pass C, local
        k_fft01<MODE_INV, 6><<<g01, c->fft01_threads, c->smem01, c->stream>>>(c->field[r], none, none, nop, Gl, c->Tl, c->fft01_ncomp, 0.0, c->ctl);
        c->launches++;
    }
    for (int r = 0; r < P; r++) {                        // halo 2: X of the first slice of rank r+1 -> rank r
        const int q = (r + 1) % P;
        slab_exchange(c, "X halo", c->halo_x[r], (size_t)c->S * sizeof(cplx), c->field[q], (size_t)c->Vl * sizeof(cplx), (size_t)c->S * sizeof(cplx), 4);
    }
    for (int r = 0; r < P; r++) {                        // S3 + S4
        if (Gl.L[0] <= 32) k_update_slab<NC, 32><<<(unsigned)(c->Vl / 32), 128, 0, c->stream>>>(c->links[r], c->field[r], c->halo_x[r], Gl, half_alpha, c->ctl, r == 0);
        else k_update_slab<NC, 64><<<(unsigned)(c->Vl / 64), 256, 0, c->stream>>>(c->links[r], c->field[r], c->halo_x[r], Gl, half_alpha, c->ctl, r == 0);
        c->launches++;
    }
}

lgf_status slab_run(lgf_slab_ctx* c, double alpha, double tol, int max_iter, bool poll) {
    lgf_status st = slab_reset_ctl(c, tol, max_iter);
    if (st != LGF_OK) return st;
    c->copy_err = cudaSuccess; c->copy_what = "";
    long long left = (long long)max_iter + 1;
    while (left > 0) {
        const int nb = (int)(left < 8 ? left : 8);
        for (int i = 0; i < nb; i++) { if (c->NC == 6) slab_body<6>(c, 0.5 * alpha); else slab_body<9>(c, 0.5 * alpha); }
        if (c->copy_err != cudaSuccess) {        // a halo never arrived: the links are no longer a gauge copy of the input
            char b[256];
            snprintf(b, sizeof b, "inter-rank copy (%s) failed: %s", c->copy_what, cudaGetErrorString(c->copy_err));
            c->err = b;
            cudaStreamSynchronize(c->stream); cudaGetLastError();
            c->loaded = false;
            return LGF_ERR_CUDA;
        }
        SCK(cudaGetLastError());
        left -= nb;
        if (poll || left == 0) {
            st = slab_read_ctl(c);
            if (st != LGF_OK) return st;
            if (c->h_ctl->done) break;
        }
    }
    return c->h_ctl->nonfinite ? LGF_ERR_NUMERIC : LGF_OK;
}

}  // namespace

extern "C" {

void lgf_destroy_sharded(lgf_slab_ctx* c) {
    if (!c) return;
    if (c->stream) cudaStreamSynchronize(c->stream);
    for (int r = 0; r < SLAB_MAX_RANKS; r++) if (c->ws[r]) cudaFree(c->ws[r]);
    if (c->shared) cudaFree(c->shared);
    if (c->h_ctl) cudaFreeHost(c->h_ctl);
    if (c->stream) cudaStreamDestroy(c->stream);
    delete c;
}

lgf_status lgf_create_sharded(const int dims[4], int n_ranks, lgf_storage s, lgf_slab_ctx** out) {
    g_slab_create_err.clear();                   // lgf_last_error_sharded(NULL): the text of this thread's last failed create
    auto refuse = [&](lgf_status st, const char* why) { g_slab_create_err = why; return st; };
    if (!dims || !out) return refuse(LGF_ERR_INVALID_ARG, "lgf_create_sharded: dims or out is NULL");
    *out = nullptr;
    if (s != LGF_STORE_12 && s != LGF_STORE_18) return refuse(LGF_ERR_INVALID_ARG, "lgf_create_sharded: storage is not LGF_STORE_12 or LGF_STORE_18");
    if (n_ranks < 1 || n_ranks > SLAB_MAX_RANKS || (n_ranks & (n_ranks - 1))) return refuse(LGF_ERR_INVALID_ARG, "lgf_create_sharded: n_ranks must be a power of two between 1 and 16");
    for (int k = 0; k < 4; k++) if (dims[k] < 1) return refuse(LGF_ERR_INVALID_ARG, "lgf_create_sharded: an extent is smaller than 1");
    int lg[4];
    if (!dims_ok(dims, lg)) return refuse(LGF_ERR_UNSUPPORTED, "lgf_create_sharded: extents must be powers of two, 4 <= L <= 128, L0*L1 <= 4096, L2*L3 <= 4096");
    int lgP = 0; while ((1 << lgP) < n_ranks) lgP++;
    if (lgP > lg[3] || lgP > lg[1] || dims[0] > 64)      // every rank needs a time slice and an x1 row; x0 rows of <= 64 sites
        return refuse(LGF_ERR_UNSUPPORTED, "lgf_create_sharded: n_ranks must not exceed L1 or L3, and L0 must be at most 64");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return refuse(LGF_ERR_CUDA, "lgf_create_sharded: no CUDA device (there is no CPU fallback)"); }
    lgf_slab_ctx* c = new (std::nothrow) lgf_slab_ctx();
    if (!c) return refuse(LGF_ERR_OOM, "lgf_create_sharded: host allocation of the context failed");
    c->copy_err = cudaSuccess; c->copy_what = "";
    c->P = n_ranks; c->lgP = lgP; c->NC = (s == LGF_STORE_12) ? 6 : 9;
    for (int r = 0; r < SLAB_MAX_RANKS; r++) c->ws[r] = nullptr;
    c->shared = nullptr; c->h_ctl = nullptr; c->stream = nullptr; c->loaded = false; c->launches = 0; c->copies = 0;
    slab_geom(c->Gg, lg[0], lg[1], lg[2], lg[3], 4);
    slab_geom(c->Gl, lg[0], lg[1], lg[2], lg[3] - lgP, 4);
    slab_geom(c->Gt, lg[0], lg[1] - lgP, lg[2], lg[3], 4);
    c->Vl = c->Gl.V; c->S = 1LL << c->Gl.sh[3];
    c->nb = (int)(c->Vl / 128);
    auto fail = [&](lgf_status st) {
        const cudaError_t e = cudaGetLastError();
        g_slab_create_err = !c->err.empty() ? c->err
            : st == LGF_ERR_OOM ? std::string("lgf_create_sharded: device or pinned-host allocation failed")
            : st == LGF_ERR_UNSUPPORTED ? std::string("lgf_create_sharded: a rank's slab is too small (< 128 sites) or its FFT tile exceeds shared memory")
            : std::string("lgf_create_sharded: CUDA set-up failed") + (e != cudaSuccess ? std::string(": ") + cudaGetErrorString(e) : std::string());
        lgf_destroy_sharded(c);
        return st;
    };
    if (c->nb < 1) return fail(LGF_ERR_UNSUPPORTED);
    if (cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) != cudaSuccess) return fail(LGF_ERR_CUDA);
    // per-rank workspaces
    const size_t b_links = align_up((size_t)c->Vl * 4 * c->NC * sizeof(cplx), 256), b_field = align_up((size_t)c->Vl * 4 * sizeof(cplx), 256);
    const size_t b_hu = align_up((size_t)c->S * c->NC * sizeof(cplx), 256), b_hx = align_up((size_t)c->S * 4 * sizeof(cplx), 256);
    for (int r = 0; r < n_ranks; r++) {
        if (cudaMalloc(&c->ws[r], b_links + 2 * b_field + b_hu + b_hx) != cudaSuccess) { cudaGetLastError(); return fail(LGF_ERR_OOM); }
        char* p = c->ws[r];
        c->links[r] = reinterpret_cast<cplx*>(p); p += b_links;
        c->field[r] = reinterpret_cast<cplx*>(p); p += b_field;
        c->fieldT[r] = reinterpret_cast<cplx*>(p); p += b_field;
        c->halo_u[r] = reinterpret_cast<cplx*>(p); p += b_hu;
        c->halo_x[r] = reinterpret_cast<cplx*>(p);
    }
    // shared: partials, control block, history, tables
    const size_t b_part = align_up((size_t)n_ranks * c->nb * 16, 256), b_ctl = align_up(sizeof(Ctl), 256), b_hist = align_up((size_t)HIST_CAP * 16, 256);
    const size_t b_tab = align_up(4 * 128 * 16 + 4 * 128 * 8, 256);
    if (cudaMalloc(&c->shared, b_part + b_ctl + b_hist + b_tab) != cudaSuccess) { cudaGetLastError(); return fail(LGF_ERR_OOM); }
    c->partials = reinterpret_cast<double2*>(c->shared);
    c->ctl = reinterpret_cast<Ctl*>(c->shared + b_part);
    c->hist = reinterpret_cast<double2*>(c->shared + b_part + b_ctl);
    char* tb = c->shared + b_part + b_ctl + b_hist;
    if (cudaHostAlloc(&c->h_ctl, sizeof(Ctl), cudaHostAllocDefault) != cudaSuccess) return fail(LGF_ERR_OOM);
    // tables of the whole lattice (as build_tables)
    {
        std::vector<real> tw(4 * 128 * 2, real(0));
        std::vector<double> sv(4 * 128, 0.0);
        const long double pi = 3.141592653589793238462643383279502884L;
        for (int mu = 0; mu < 4; mu++) {
            c->Tl.plan[mu] = make_plan(lg[mu], (mu & 1) != 0, false);      // the generic passes: plans without the 64-point pass-B exception
            const int L = dims[mu];
            for (int k = 0; k < L; k++) {
                long double a = 2.0L * pi * (long double)k / (long double)L;
                double cr = (double)cosl(a), sr = (double)sinl(a);
                if ((4 * k) % L == 0) { const int q = 4 * k / L; const double cc[4] = {1, 0, -1, 0}, ss[4] = {0, 1, 0, -1}; cr = cc[q]; sr = ss[q]; }
                tw[(mu * 128 + k) * 2] = (real)cr; tw[(mu * 128 + k) * 2 + 1] = (real)(-sr);
            }
            for (int p = 0; p < L; p++) {
                const int n = stored_freq(p, lg[mu], c->Tl.plan[mu]);
                long double sn = sinl(pi * (long double)n / (long double)L);
                sv[mu * 128 + p] = (n == 0) ? 0.0 : (double)(4.0L * sn * sn);
            }
        }
        if (cudaMemcpyAsync(tb, tw.data(), tw.size() * sizeof(real), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
            cudaMemcpyAsync(tb + 4 * 128 * 16, sv.data(), sv.size() * 8, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
            cudaStreamSynchronize(c->stream) != cudaSuccess) return fail(LGF_ERR_CUDA);
        for (int mu = 0; mu < 4; mu++) {
            c->Tl.tw[mu] = reinterpret_cast<const cplx*>(tb) + mu * 128;
            c->Tl.s[mu] = reinterpret_cast<const double*>(tb + 4 * 128 * 16) + mu * 128;
        }
        for (int r = 0; r < n_ranks; r++) { c->Tt[r] = c->Tl; c->Tt[r].s[1] = c->Tl.s[1] + r * c->Gt.L[1]; }
    }
    // launch parameters of the generic passes (as setup_kernels) on the local and the transposed lattice
    {
        const Geom& G = c->Gl;
        auto smem01 = [&](int ncomp) { return (size_t)((G.L[0] + 1) * G.L[1] * ncomp + G.L[0] + G.L[1]) * sizeof(cplx); };
        int ncomp = 4;
        while (ncomp > 1 && smem01(ncomp) > 100 * 1024) ncomp >>= 1;
        c->fft01_ncomp = ncomp; c->smem01 = smem01(ncomp);
        int th = G.L[0] * G.L[1] * 4 / 8; if (th > 256) th = 256; if (th < 32) th = 32;
        c->fft01_threads = th;
        const Geom& H = c->Gt;
        const int n23 = H.L[2] * H.L[3];
        int lgC = 3; if (lgC > H.lg[0]) lgC = H.lg[0];
        while (lgC > 1 && ((size_t)n23 << lgC) * 16 > 64 * 1024) lgC--;
        if (((size_t)n23 << lgC) * 16 > (size_t)MAX_SMEM - 8192) lgC = 0;
        c->fft23_lgC = lgC;
        const int C0 = 1 << lgC;
        c->fft23_S2 = C0 * H.L[2] + (C0 < 8 ? C0 : 0);
        c->smem23 = (size_t)(c->fft23_S2 * H.L[3] + H.L[2] + H.L[3]) * sizeof(cplx) + (size_t)(H.L[2] + H.L[3]) * 8;
        if (c->smem23 > (size_t)MAX_SMEM || c->smem01 > (size_t)MAX_SMEM) return fail(LGF_ERR_UNSUPPORTED);
        th = (n23 << lgC) / 8; if (th > 256) th = 256; if (th < 32) th = 32;
        c->fft23_threads = th;
        if (set_smem(k_fft01<MODE_FWD, 6>, c->smem01) != cudaSuccess || set_smem(k_fft01<MODE_INV, 6>, c->smem01) != cudaSuccess ||
            set_smem(k_fft23_mid, c->smem23) != cudaSuccess) return fail(LGF_ERR_CUDA);
    }
    if (slab_reset_ctl(c, -1.0, 0) != LGF_OK) return fail(LGF_ERR_CUDA);
    *out = c;
    return LGF_OK;
}

int lgf_sharded_ranks(lgf_slab_ctx* c) { return c ? c->P : 0; }

// Rank r's slab is the contiguous range [r Vl, (r+1) Vl) of the canonical array (x3 is the slowest index).
lgf_status lgf_load_links_sharded(lgf_slab_ctx* c, const double* host_links) {
    if (!c || !host_links) return LGF_ERR_INVALID_ARG;
    dcplx* tmp = nullptr;
    if (cudaMalloc(&tmp, (size_t)c->Vl * 576) != cudaSuccess) { cudaGetLastError(); return LGF_ERR_OOM; }
    lgf_status st = LGF_OK;
    for (int r = 0; r < c->P && st == LGF_OK; r++) {
        if (cudaMemcpyAsync(tmp, host_links + (size_t)r * c->Vl * 72, (size_t)c->Vl * 576, cudaMemcpyHostToDevice, c->stream) != cudaSuccess) { st = LGF_ERR_CUDA; break; }
        const unsigned grid = (unsigned)((c->Vl * 4 + 255) / 256);
        if (c->NC == 6) k_layout_in<6><<<grid, 256, 0, c->stream>>>(tmp, c->links[r], c->Vl, 0, c->Vl, 9);
        else k_layout_in<9><<<grid, 256, 0, c->stream>>>(tmp, c->links[r], c->Vl, 0, c->Vl, 9);
        c->launches++;
    }
    if (cudaStreamSynchronize(c->stream) != cudaSuccess || cudaGetLastError() != cudaSuccess) st = LGF_ERR_CUDA;
    cudaFree(tmp);
    if (st == LGF_OK) c->loaded = true;
    return st;
}
lgf_status lgf_get_links_sharded(lgf_slab_ctx* c, double* host_links) {
    if (!c || !host_links) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    dcplx* tmp = nullptr;
    if (cudaMalloc(&tmp, (size_t)c->Vl * 576) != cudaSuccess) { cudaGetLastError(); return LGF_ERR_OOM; }
    lgf_status st = LGF_OK;
    for (int r = 0; r < c->P && st == LGF_OK; r++) {
        const unsigned grid = (unsigned)((c->Vl * 4 + 255) / 256);
        if (c->NC == 6) k_layout_out<6><<<grid, 256, 0, c->stream>>>(c->links[r], tmp, c->Vl, 0, c->Vl, 9);
        else k_layout_out<9><<<grid, 256, 0, c->stream>>>(c->links[r], tmp, c->Vl, 0, c->Vl, 9);
        c->launches++;
        if (cudaMemcpyAsync(host_links + (size_t)r * c->Vl * 72, tmp, (size_t)c->Vl * 576, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) st = LGF_ERR_CUDA;
    }
    if (cudaStreamSynchronize(c->stream) != cudaSuccess || cudaGetLastError() != cudaSuccess) st = LGF_ERR_CUDA;
    cudaFree(tmp);
    return st;
}

lgf_status lgf_iterate_sharded(lgf_slab_ctx* c, int n, double alpha, double* F, double* theta) {
    if (!c || n < 0 || !(alpha > 0.0) || !std::isfinite(alpha)) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    lgf_status st = slab_run(c, alpha, -1.0, n, false);
    if (st != LGF_OK) return st;
    if (F) *F = c->h_ctl->F;
    if (theta) *theta = c->h_ctl->theta;
    return LGF_OK;
}
lgf_status lgf_fix_sharded(lgf_slab_ctx* c, double alpha, double theta_tol, int max_iter, int* n_iter, double* F, double* theta) {
    if (!c || max_iter < 0 || !(alpha > 0.0) || !std::isfinite(alpha) || !(theta_tol >= 0.0)) return LGF_ERR_INVALID_ARG;
    if (!c->loaded) return LGF_ERR_NOT_LOADED;
    lgf_status st = slab_run(c, alpha, theta_tol, max_iter, true);
    if (st != LGF_OK) return st;
    if (n_iter) *n_iter = c->h_ctl->iters;
    if (F) *F = c->h_ctl->F;
    if (theta) *theta = c->h_ctl->theta;
    return c->h_ctl->converged ? LGF_OK : LGF_NOT_CONVERGED;
}
lgf_status lgf_get_history_sharded(lgf_slab_ctx* c, double* hist, int capacity, int* n_out) {
    if (!c || !hist || capacity < 0 || !n_out) return LGF_ERR_INVALID_ARG;
    int n = c->h_ctl->n_meas; if (n > HIST_CAP) n = HIST_CAP; if (n > capacity) n = capacity;
    if (n > 0) {
        SCK(cudaMemcpyAsync(hist, c->hist, (size_t)n * 16, cudaMemcpyDeviceToHost, c->stream));
        SCK(cudaStreamSynchronize(c->stream));
    }
    *n_out = n;
    return LGF_OK;
}
// Bytes one rank SENDS per iteration: [0] halo 1 (U_3 slice), [1] halo 2 (X slice), [2] the two transposes (the part of
// its field that changes owner, twice); [3] kernels launched and [4] inter-rank copies issued so far (all ranks).
lgf_status lgf_sharded_traffic(lgf_slab_ctx* c, long long out[5]) {
    if (!c || !out) return LGF_ERR_INVALID_ARG;
    out[0] = c->S * c->NC * (long long)sizeof(cplx);
    out[1] = c->S * 4 * (long long)sizeof(cplx);
    out[2] = 2 * (c->Vl * 4 * (long long)sizeof(cplx)) * (c->P - 1) / c->P;
    out[3] = c->launches;
    out[4] = c->copies;
    return LGF_OK;
}
const char* lgf_last_error_sharded(lgf_slab_ctx* c) { return c ? c->err.c_str() : g_slab_create_err.c_str(); }

}  // extern "C"
