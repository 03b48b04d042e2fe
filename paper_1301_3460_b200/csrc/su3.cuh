// su3.cuh -- register-level complex 3x3 algebra for the gauge-fixing kernels (fp64, sm_100a).
// Complex numbers are double2 (x = re, y = im).  Everything is __forceinline__ so that unused rows
// and entries are dead-code eliminated in each kernel.
// Precision: the translation unit defines LGF_F32 for the fp32 build (real = float, cplx = float2, namespace renamed by
// "#define lgf lgf32" in lgf_api.cu); default fp64.  Sums over the lattice (theta, F) and the p^2 filter weights stay
// double in both builds.
#pragma once
#include <cuda_runtime.h>

namespace lgf {

#ifdef LGF_F32
typedef float real;
typedef float2 cplx;
#else
typedef double real;
typedef double2 cplx;
#endif
typedef double2 dcplx;      // host-facing complex (the C ABI speaks double in every precision)

__device__ __forceinline__ cplx mk(real a, real b) { cplx r; r.x = a; r.y = b; return r; }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mk(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return mk(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cconj(cplx a) { return mk(a.x, -a.y); }
__device__ __forceinline__ cplx cscale(cplx a, real s) { return mk(a.x * s, a.y * s); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) { return mk(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
// conj(a) * b
__device__ __forceinline__ cplx ccmul(cplx a, cplx b) { return mk(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }
// c + a*b
__device__ __forceinline__ cplx cfma(cplx a, cplx b, cplx c) {
    return mk(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}
// c + a*conj(b)
__device__ __forceinline__ cplx cfmac(cplx a, cplx b, cplx c) {
    return mk(fma(a.x, b.x, fma(a.y, b.y, c.x)), fma(a.y, b.x, fma(-a.x, b.y, c.y)));
}
// c - a*b
__device__ __forceinline__ cplx cfnma(cplx a, cplx b, cplx c) {
    return mk(fma(-a.x, b.x, fma(a.y, b.y, c.x)), fma(-a.x, b.y, fma(-a.y, b.x, c.y)));
}
__device__ __forceinline__ real cnorm2(cplx a) { return fma(a.x, a.x, a.y * a.y); }

// Row 2 of a special unitary matrix from rows 0,1: row2 = conj(row0 x row1)  ("12 real
// number representation").  u[0..2] = row 0, u[3..5] = row 1, u[6..8] = row 2.
__device__ __forceinline__ void third_row(cplx (&u)[9]) {
    u[6] = cconj(cfnma(u[2], u[4], cmul(u[1], u[5])));
    u[7] = cconj(cfnma(u[0], u[5], cmul(u[2], u[3])));
    u[8] = cconj(cfnma(u[1], u[3], cmul(u[0], u[4])));
}

// 128-bit loads/stores of one complex double
__device__ __forceinline__ cplx ldg2(const cplx* p) { return __ldg(p); }

// field (Delta~ / X~ / X) accesses: ld_field where the same kernel later overwrites the location (plain load),
// ldc_field where the field is read-only for the kernel (non-coherent path)
__device__ __forceinline__ cplx ld_field(const cplx* p) { return *p; }
__device__ __forceinline__ cplx ldc_field(const cplx* p) { return __ldg(p); }
__device__ __forceinline__ void st_field(cplx* p, cplx v) { *p = v; }

// Line prefetch into L2 (no destination register): used to pull a thread's NEXT site towards the SM while it works on
// the current one, so that the later loads see L2 latency instead of DRAM latency.
__device__ __forceinline__ void prefetch_line_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// true for one lane per 128-byte line of consecutive complex numbers (lanes run over consecutive sites)
#ifndef LGF_PF_ONE_PER_LINE
#define LGF_PF_ONE_PER_LINE 0
#endif
__device__ __forceinline__ bool prefetch_lane() {
    return !LGF_PF_ONE_PER_LINE || (threadIdx.x & (128 / (int)sizeof(cplx) - 1)) == 0;
}

// Load link (x, mu) from the structure-of-arrays store: entry c of direction mu is the V-array at
// links + (mu*NC + c)*V, NC = 6 (12-real: rows 0,1) or 9 (18-real).  Row 2 is rebuilt for NC = 6.
// RO = true: the links are read-only for the whole kernel (S1, read-outs): non-coherent loads (ld.global.nc).
// RO = false: the kernel also writes the links (the in-place update kernels): plain loads, as ld.global.nc is specified
// for data nobody writes during the kernel's lifetime.
template <int NC, bool RO = true>
__device__ __forceinline__ void load_link(const cplx* links, long long V, int mu, long long x, cplx (&u)[9]) {
    const cplx* p = links + (long long)(mu * NC) * V + x;
#pragma unroll
    for (int c = 0; c < NC; c++) u[c] = RO ? __ldg(p + (long long)c * V) : p[(long long)c * V];
    if (NC == 6) third_row(u);
}
template <int NC>
__device__ __forceinline__ void store_link(cplx* links, long long V, int mu, long long x, const cplx (&u)[9]) {
    cplx* p = links + (long long)(mu * NC) * V + x;
#pragma unroll
    for (int c = 0; c < NC; c++) p[(long long)c * V] = u[c];
}

// S3: g = rowGramSchmidt(M), M = 1 + (alpha/2) X, X given by its packed independent components
//   f0 = X01, f1 = X02, f2 = X12, f3 = (Im X00, Im X11);  X_ji = -conj(X_ij), X anti-Hermitian traceless.
// Only rows 0 and 1 of M enter; row 2 of g is conj(u x v).  ha = alpha/2.   [north_star step 3]
__device__ __forceinline__ void build_g(cplx f0, cplx f1, cplx f2, cplx f3, real ha, cplx (&g)[9]) {
    cplx m00 = mk(real(1), ha * f3.x), m01 = cscale(f0, ha), m02 = cscale(f1, ha);
    cplx m10 = mk(-ha * f0.x, ha * f0.y), m11 = mk(real(1), ha * f3.y), m12 = cscale(f2, ha);
    real n0 = cnorm2(m00) + cnorm2(m01) + cnorm2(m02);
    real r0 = real(1) / sqrt(n0);
    g[0] = cscale(m00, r0); g[1] = cscale(m01, r0); g[2] = cscale(m02, r0);
    // <u, M1> = sum_j conj(u_j) M1_j
    cplx ip = ccmul(g[0], m10);
    ip = cadd(ip, ccmul(g[1], m11));
    ip = cadd(ip, ccmul(g[2], m12));
    cplx v0 = cfnma(ip, g[0], m10), v1 = cfnma(ip, g[1], m11), v2 = cfnma(ip, g[2], m12);
    real n1 = cnorm2(v0) + cnorm2(v1) + cnorm2(v2);
    real r1 = real(1) / sqrt(n1);
    g[3] = cscale(v0, r1); g[4] = cscale(v1, r1); g[5] = cscale(v2, r1);
    third_row(g);
}

// S4 for one link: r = g * U * gp^dag.  NROWS = 2 computes rows 0,1 only (12-real storage).
template <int NROWS>
__device__ __forceinline__ void rotate_link(const cplx (&g)[9], const cplx (&u)[9], const cplx (&gp)[9], cplx (&r)[9]) {
#pragma unroll
    for (int i = 0; i < NROWS; i++) {
        cplx t[3];
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cplx s = cmul(g[3 * i + 0], u[j]);
            s = cfma(g[3 * i + 1], u[3 + j], s);
            s = cfma(g[3 * i + 2], u[6 + j], s);
            t[j] = s;
        }
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cplx s = cmulc(t[0], gp[3 * j + 0]);
            s = cfmac(t[1], gp[3 * j + 1], s);
            s = cfmac(t[2], gp[3 * j + 2], s);
            r[3 * i + j] = s;
        }
    }
}

// S2b filter weight scale / p2 (scale = p2max / V), 0 for the zero mode.  p2 lies in [4 sin^2(pi/128), 16]: no special
// cases, so the division is a reciprocal seed (MUFU.RCP64H, ~20 bits) and two Newton steps -- within 2 ulp of the IEEE
// quotient at a quarter of its instructions (the IEEE fp64 division was a quarter of pass B's instruction stream).
// Every pass-B kernel, generic or compile-time-sized, takes the weight from this one function.  Its argument is not summed
// in one order everywhere (k_tb_mid forms p2 as ((s0+s1)+s2)+s3, k_fft23_mid as (s0+s1)+(s2+s3)), so two kernel
// selections can differ in the last bit of p2 and hence of the weight: they agree to rounding, not bit for bit (the
// parity tests bound X at 1e-13 relative for every selection).
__device__ __forceinline__ double filter_weight(double scale, double p2) {
    if (!(p2 > 0.0)) return 0.0;
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(p2));
    double e = fma(-p2, r, 1.0);
    r = fma(r, e, r);
    e = fma(-p2, r, 1.0);
    r = fma(r, e, r);
    return scale * r;
}

// Lattice geometry: every L_mu is a power of two, x = x0 + L0*(x1 + L1*(x2 + L2*x3)).
struct Geom {
    int L[4];
    int lg[4];    // log2 L
    int sh[4];    // log2 stride of axis mu (sum of lg of lower axes)
    int nd;       // directions in the gauge condition: 4 Landau (the paper), 3 Coulomb (mu = 0..2)
    long long V;
};
__device__ __forceinline__ int coord(const Geom& G, long long x, int mu) { return (int)(x >> G.sh[mu]) & (G.L[mu] - 1); }
__device__ __forceinline__ long long fwd(const Geom& G, long long x, int mu) {
    int c = coord(G, x, mu);
    return (c == G.L[mu] - 1) ? x - ((long long)(G.L[mu] - 1) << G.sh[mu]) : x + (1LL << G.sh[mu]);
}
__device__ __forceinline__ long long bwd(const Geom& G, long long x, int mu) {
    int c = coord(G, x, mu);
    return (c == 0) ? x + ((long long)(G.L[mu] - 1) << G.sh[mu]) : x - (1LL << G.sh[mu]);
}

// Programmatic dependent launch (sm_90+): every kernel of the iteration is launched with the programmatic-serialization
// attribute and waits on the device for the complete, flushed end of its predecessor (griddepcontrol.wait) before it
// touches global memory -- so stream order is kept, and what overlaps is the launch latency of kernel n+1 with the tail
// of kernel n.  An explicit early trigger (griddepcontrol.launch_dependents at kernel entry, LGF_PDL_EARLY_TRIGGER = 1)
// lets the successor's CTAs become resident while the predecessor's last wave still runs; measured on B200 that is
// slower (311.9 against 307.7 us per iteration at 32^4, 27.0 against 24.5 us at 16^4: the waiting CTAs hold registers
// and shared memory), so the trigger is left implicit at kernel exit.  No-ops when the launch does not carry the
// attribute.
#ifndef LGF_PDL_EARLY_TRIGGER
#define LGF_PDL_EARLY_TRIGGER 0
#endif
__device__ __forceinline__ void pdl_enter() {
    if (LGF_PDL_EARLY_TRIGGER) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// Device-resident control block shared by all kernels of one context.
struct Ctl {
    double F, theta;       // last measurement (S1)
    double theta_tol;      // S5: stop when theta < theta_tol; negative = never
    int max_iter;          // stop after this many updates
    int done;              // 1: every later kernel exits at once, the link state is frozen
    int converged;         // 1: stopped by theta < theta_tol
    int iters;             // link updates applied so far
    int nonfinite;         // theta or F not finite
    int n_meas;            // measurements made (index into the history)
    int hist_cap;
    // stagnation guard (the fp32 phase of LGF_MIXED): stop when theta has not halved within stall_window measurements
    int stall_window;      // 0: off
    int stall_count;       // measurements since theta last fell below half of theta_mark
    int stalled;           // 1: stopped by the guard
    double theta_mark;
};

}  // namespace lgf
