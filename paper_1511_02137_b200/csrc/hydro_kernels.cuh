// hydro_kernels.cuh -- device code of the hot path (sm_100a).  PRODUCT; shares nothing with oracle/.
//
// Steps of SURVEY.md 8(a) / DESIGN.md "Kernels":
//   k_prim        a-1 con2prim (p = e/3 closed form, admissibility cap R9) + a-2 wavespeeds and their global max
//   k_sweep<DIR>  a-3 WENO7 reconstruction of the Lax-Friedrichs split fluxes along DIR, a-4 flux divergence,
//                 a-7 outflow ghosts by index clamping; the last sweep also does a-6 (SSP-RK3 stage combination)
//   k_source      a-5 jet point source (eq. 2, 3 of the paper) + diagnostics bookkeeping
//
// The WENO7 arithmetic is organised for the FP64 pipe, which bounds this path:
// every thread marches along the sweep axis and keeps a sliding window of undivided differences of the split
// flux in registers, so each new cell costs 4 subtractions + 1 FMA-pair per split sign, the four smoothness
// indicators are sums of three squares built from those differences ("7th order WENO"; the
// formulas are derived in DESIGN.md "WENO7 in difference form"), the four nonlinear weights share one common
// denominator, and the left- and right-biased reconstructions of an interface share ONE reciprocal.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace hydro_dev {

constexpr int MAX_JETS = 64;

// ------------------------------------------------------------------------------------------------ diagnostics
// One slot per "generation" of primitives (two alternate): k_prim fills a slot for the state it converts,
// k_source commits it to the totals when a stage actually consumes that state.
struct DiagSlot {
    unsigned long long alpha_bits[3];   // max wavespeed per direction, as the bit pattern of a non-negative real
    unsigned long long ncap;            // cells where the floor / cap of con2prim fired
    unsigned long long nan_flag;        // a non-finite conserved value was seen
    unsigned long long pad[3];
};
struct Diag {
    DiagSlot slot[2];
    unsigned long long ncap_total;
    unsigned long long nan_total;
    double alpha_last[3];               // alpha of the last evaluated stage
    double deposited[4];                // jets: total (E, Mx, My, Mz) deposited [GeV]
    double last_q[3][MAX_JETS];         // q^s of every jet in the stages of the last step
};

struct JetDev {
    double x0, y0, z0, nx, ny, nz, k_rad, k_coll, crcf;
    long long step_added;
};

// ------------------------------------------------------------------------------------------------ real traits
template <typename R> struct Real;
template <> struct Real<double> {
    typedef unsigned long long bits_t;
    static __device__ __forceinline__ unsigned long long to_bits(double x) { return (unsigned long long)__double_as_longlong(x); }
    static __device__ __forceinline__ double from_bits(unsigned long long b) { return __longlong_as_double((long long)b); }
    static __device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
    static __device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
    // reciprocal to ~1 ulp for normal, well-scaled arguments: hardware seed + two Newton steps
    static __device__ __forceinline__ double rcp_(double x) {
        double r;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
        double e = fma(-x, r, 1.0);
        r = fma(r, e, r);
        e = fma(-x, r, 1.0);
        r = fma(r, e, r);
        return r;
    }
    // 1/x and sqrt(x) for normal, positive, well-scaled x without the special-case paths of the IEEE routines
    // (error <= ~1 ulp): hardware seeds (upper 32 bits, ~2^-20) + Newton-type corrections.
    static __device__ __forceinline__ double rcp_fast(double x) {
        double r;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
        const double e = fma(-x, r, 1.0);
        r = fma(r, fma(e, e, e), r);                    // cubic step: error e^3
        return fma(r, fma(-x, r, 1.0), r);              // + one linear step: last-bit accuracy
    }
    static __device__ __forceinline__ double sqrt_fast(double x) {
        double y;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        double g = x * y, h = 0.5 * y;                  // g ~ sqrt(x), h ~ 1/(2 sqrt(x))
        double r = fma(-g, h, 0.5);
        g = fma(g, r, g);
        h = fma(h, r, h);
        r = fma(-g, h, 0.5);
        g = fma(g, r, g);
        h = fma(h, r, h);
        return fma(fma(-g, g, x), h, g);                // final residual correction
    }
};
template <> struct Real<float> {
    typedef unsigned int bits_t;
    static __device__ __forceinline__ unsigned long long to_bits(float x) { return (unsigned long long)__float_as_uint(x); }
    static __device__ __forceinline__ float from_bits(unsigned long long b) { return __uint_as_float((unsigned int)b); }
    static __device__ __forceinline__ float sqrt_(float x) { return sqrtf(x); }
    static __device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
    static __device__ __forceinline__ float rcp_(float x) { return 1.0f / x; }
    static __device__ __forceinline__ float rcp_fast(float x) { return 1.0f / x; }
    static __device__ __forceinline__ float sqrt_fast(float x) { return sqrtf(x); }
};

// ------------------------------------------------------------------------------------------------ a-1, a-2
// con2prim for p = e/3 (eq. 1 with u^mu = gamma(1,v);  e^2 + 2Ee - 3(E^2 - M^2) = 0), reading R9:
// E floored, |M| capped at (1-delta)E, stored U untouched.  Outputs p and wt = scale/(E+p) so that the
// velocity used by every flux is v_d = M_d * wt with the STORED momentum M_d.
template <typename R>
__device__ __forceinline__ void con2prim(R E, R Mx, R My, R Mz, R e_floor, R one_minus_delta, R& p, R& wt,
                                         int& limited) {
    typedef Real<R> T;
    limited = 0;
    if (E < e_floor) { E = e_floor; limited = 1; }
    R M2 = Mx * Mx + My * My + Mz * Mz;
    const R cap = one_minus_delta * E;
    R sc = R(1);
    if (M2 > cap * cap) {                                            // rare: |M| > (1 - delta) E
        sc = cap / T::sqrt_(M2);
        limited = 1;
        const R mx = Mx * sc, my = My * sc, mz = Mz * sc;
        M2 = mx * mx + my * my + mz * mz;
    }
    const R s = T::sqrt_fast(R(4) * E * E - R(3) * M2);
    const R e = R(3) * (E * E - M2) * T::rcp_fast(E + s);
    p = e * R(1.0 / 3.0);
    wt = sc * T::rcp_fast(E + p);
}

// max(|lambda_+|, |lambda_-|) of the acoustic eigenvalues along a direction with velocity component vd:
// lambda = [vd (1-cs2) +- cs sqrt((1-v2)(1 - v2 cs2 - vd^2 (1-cs2)))] / (1 - v2 cs2),  cs2 = 1/3;
// root >= 0 and den > 0, so the larger modulus is (|vd| (1-cs2) + root) / den.
template <typename R>
__device__ __forceinline__ R max_wavespeed(R vd, R den, R inv_den, R om_v2) {
    const R cs2 = R(1.0 / 3.0);
    R rad = om_v2 * (den - vd * vd * (R(1) - cs2));
    rad = rad < R(1e-30) ? R(1e-30) : rad;                           // clamp (R9); keeps the rsqrt seed finite
    const R root = R(0.57735026918962576451) * Real<R>::sqrt_fast(rad);
    R a = vd * (R(1) - cs2);
    a = a < R(0) ? -a : a;
    return (a + root) * inv_den;
}

template <typename R>
struct PrimArgs {
    const R* U;        // nf blocks of N
    R* P;              // pressure
    R* W;              // wt = scale/(E+p)
    Diag* diag;
    int slot;
    long long N;
    R e_floor, one_minus_delta;
};

template <typename R>
__global__ void __launch_bounds__(256) k_prim(PrimArgs<R> a) {
    R am[3] = {R(0), R(0), R(0)};
    unsigned int ncap = 0, bad = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    auto cell = [&](long long c, R E, R Mx, R My, R Mz) {
        R p, wt;
        int lim;
        con2prim<R>(E, Mx, My, Mz, a.e_floor, a.one_minus_delta, p, wt, lim);
        a.P[c] = p;
        a.W[c] = wt;
        ncap += lim;
        // finite check: x - x is 0 for finite x, NaN otherwise
        R chk = (E - E) + (Mx - Mx) + (My - My) + (Mz - Mz);
        bad |= (chk == R(0)) ? 0u : 1u;
        R vx = Mx * wt, vy = My * wt, vz = Mz * wt;
        R v2 = vx * vx + vy * vy + vz * vz;
        R om = R(1) - v2;
        om = om < R(0) ? R(0) : om;
        const R den = R(1) - v2 * R(1.0 / 3.0);
        const R inv_den = Real<R>::rcp_fast(den);
        R lx = max_wavespeed<R>(vx, den, inv_den, om);
        R ly = max_wavespeed<R>(vy, den, inv_den, om);
        R lz = max_wavespeed<R>(vz, den, inv_den, om);
        am[0] = lx > am[0] ? lx : am[0];
        am[1] = ly > am[1] ? ly : am[1];
        am[2] = lz > am[2] ? lz : am[2];
    };
    // two cells per trip: eight independent loads in flight per thread before the arithmetic starts
    long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; c + stride < a.N; c += 2 * stride) {
        const long long c2 = c + stride;
        const R E = a.U[c], Mx = a.U[a.N + c], My = a.U[2 * a.N + c], Mz = a.U[3 * a.N + c];
        const R E2 = a.U[c2], Mx2 = a.U[a.N + c2], My2 = a.U[2 * a.N + c2], Mz2 = a.U[3 * a.N + c2];
        cell(c, E, Mx, My, Mz);
        cell(c2, E2, Mx2, My2, Mz2);
    }
    if (c < a.N) cell(c, a.U[c], a.U[a.N + c], a.U[2 * a.N + c], a.U[3 * a.N + c]);
    // warp reduction by shuffles, then one atomic per warp on the bit pattern (non-negative reals order like
    // unsigned integers; the max is exact, hence order independent)
    unsigned long long ab[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) ab[d] = Real<R>::to_bits(am[d]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            unsigned long long o = __shfl_xor_sync(0xffffffffu, ab[d], off);
            ab[d] = o > ab[d] ? o : ab[d];
        }
        ncap += __shfl_xor_sync(0xffffffffu, ncap, off);
        bad |= __shfl_xor_sync(0xffffffffu, bad, off);
    }
    __shared__ unsigned long long sm[8][5];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sm[warp][0] = ab[0]; sm[warp][1] = ab[1]; sm[warp][2] = ab[2]; sm[warp][3] = ncap; sm[warp][4] = bad; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long r[5] = {0, 0, 0, 0, 0};
        const int nw = blockDim.x >> 5;
        for (int w = 0; w < nw; ++w) {
            for (int d = 0; d < 3; ++d) r[d] = sm[w][d] > r[d] ? sm[w][d] : r[d];
            r[3] += sm[w][3];
            r[4] |= sm[w][4];
        }
        DiagSlot* s = &a.diag->slot[a.slot];
        for (int d = 0; d < 3; ++d) atomicMax(&s->alpha_bits[d], r[d]);
        if (r[3]) atomicAdd(&s->ncap, r[3]);
        if (r[4]) atomicOr(&s->nan_flag, 1ull);
    }
}

// primitives for hydro_get_fields(which = 1): (e, vx, vy, vz [, n])
template <typename R>
__global__ void __launch_bounds__(256) k_prims_out(const R* __restrict__ U, R* __restrict__ out, long long N, int nf,
                                                   R e_floor, R one_minus_delta) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += stride) {
        R E = U[c], Mx = U[N + c], My = U[2 * N + c], Mz = U[3 * N + c];
        R p, wt;
        int lim;
        con2prim<R>(E, Mx, My, Mz, e_floor, one_minus_delta, p, wt, lim);
        R vx = Mx * wt, vy = My * wt, vz = Mz * wt;
        out[c] = R(3) * p;
        out[N + c] = vx;
        out[2 * N + c] = vy;
        out[3 * N + c] = vz;
        if (nf > 4) {
            R om = R(1) - (vx * vx + vy * vy + vz * vz);
            om = om < R(0) ? R(0) : om;
            out[4 * N + c] = U[4 * N + c] * Real<R>::sqrt_(om);
        }
    }
}

// ------------------------------------------------------------------------------------------------ a-3: WENO7
// Sliding window over seven consecutive values x_0..x_6 of one split flux, in ascending-cell order, held as
// undivided differences:  d[j] = x_{j+1}-x_j,  e[j] = d[j+1]-d[j],  third differences t_j = e[j+1]-e[j] kept
// only as s[j] = C3 t_j^2 + eps,  g[j] = t_{j+1}-t_j,  plus the last four values (the centre cell is v[0]).
template <typename R>
struct Win {
    R v[4], d[6], e[5], s[4], g[3], t;
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int j = 0; j < 4; ++j) { v[j] = R(0); s[j] = R(0); }
#pragma unroll
        for (int j = 0; j < 6; ++j) d[j] = R(0);
#pragma unroll
        for (int j = 0; j < 5; ++j) e[j] = R(0);
#pragma unroll
        for (int j = 0; j < 3; ++j) g[j] = R(0);
        t = R(0);
    }
    __device__ __forceinline__ void push(R x, R c3, R eps) {
        R dn = x - v[3];
        R en = dn - d[5];
        R tn = en - e[4];
        R gn = tn - t;
        R sn = Real<R>::fma_(c3 * tn, tn, eps);
        v[0] = v[1]; v[1] = v[2]; v[2] = v[3]; v[3] = x;
        d[0] = d[1]; d[1] = d[2]; d[2] = d[3]; d[3] = d[4]; d[4] = d[5]; d[5] = dn;
        e[0] = e[1]; e[1] = e[2]; e[2] = e[3]; e[3] = e[4]; e[4] = en;
        s[0] = s[1]; s[1] = s[2]; s[2] = s[3]; s[3] = sn;
        g[0] = g[1]; g[1] = g[2]; g[2] = gn;
        t = tn;
    }
};

// One WENO7-JS reconstruction (r = 4) at the face between x_3 and x_4 (MIR = false, left-biased, centre x_3)
// or of the mirrored data (MIR = true: the window holds x_0..x_6 = cells i-2..i+4, centre x_4... see below).
// With D_j, E_j, T_j, G_j the 1st..4th undivided differences in the (possibly mirrored) stencil order:
//   candidates      12 (q_0 - x_c) = 3 D_0 - 10 D_1 + 13 D_2,   12 (q_1-q_0) = 3 G_0, 12 (q_2-q_1) = -G_1,
//                   12 (q_3-q_2) = G_2
//   smoothness      36 beta_k = lam_k^2 + 39 m_k^2 + 39.05 T_k^2,
//                   lam_0 = 2 D_0 - 7 D_1 + 11 D_2, lam_1 = lam_0 + 2 G_0, lam_2 = lam_1 - G_1, lam_3 = lam_2 + 2 G_2
//                   m_0 = 2 E_1 - E_0,  m_1 = m_2 = E_2,  m_3 = 2 E_3 - E_4
//   weights         omega_k ~ d_k / (eps + beta_k)^2, d = (1, 12, 18, 4)/35 (common factors cancel)
// Returns  base12 = 12 (q_0 - x_c),  num12/den = 12 sum_k omega_k (q_k - q_0):  W = x_c + (base12 + num12/den)/12.
// For MIR the caller's window is in ascending-cell order; mirrored differences are D_j = -d[5-j], E_j = e[4-j],
// T_j^2 -> s[3-j], G_j = g[2-j].
template <typename R, bool MIR>
__device__ __forceinline__ void weno7_side(const Win<R>& w, R& base12, R& num12, R& den) {
    const R D0 = MIR ? -w.d[5] : w.d[0], D1 = MIR ? -w.d[4] : w.d[1], D2 = MIR ? -w.d[3] : w.d[2];
    const R E0 = MIR ? w.e[4] : w.e[0], E1 = MIR ? w.e[3] : w.e[1], E2 = w.e[2], E3 = MIR ? w.e[1] : w.e[3],
            E4 = MIR ? w.e[0] : w.e[4];
    const R S0 = MIR ? w.s[3] : w.s[0], S1 = MIR ? w.s[2] : w.s[1], S2 = MIR ? w.s[1] : w.s[2],
            S3 = MIR ? w.s[0] : w.s[3];
    const R G0 = MIR ? w.g[2] : w.g[0], G1 = w.g[1], G2 = MIR ? w.g[0] : w.g[2];
    typedef Real<R> T;
    R lam0 = T::fma_(R(11), D2, T::fma_(R(-7), D1, R(2) * D0));
    R lam1 = T::fma_(R(2), G0, lam0);
    R lam2 = lam1 - G1;
    R lam3 = T::fma_(R(2), G2, lam2);
    R m0 = T::fma_(R(2), E1, -E0);
    R m3 = T::fma_(R(2), E3, -E4);
    R b0 = T::fma_(lam0, lam0, T::fma_(R(39) * m0, m0, S0));
    R b1 = T::fma_(lam1, lam1, T::fma_(R(39) * E2, E2, S1));
    R b2 = T::fma_(lam2, lam2, T::fma_(R(39) * E2, E2, S2));
    R b3 = T::fma_(lam3, lam3, T::fma_(R(39) * m3, m3, S3));
    R w0, w1, w2, w3;
    if (sizeof(R) == 8) {
        // common denominator: omega_k ~ d_k prod_{j != k} (eps+beta_j)^2  (range-safe in fp64)
        R t0 = b0 * b0, t1 = b1 * b1, t2 = b2 * b2, t3 = b3 * b3;
        R p01 = t0 * t1, p23 = t2 * t3;
        w0 = t1 * p23;
        w1 = (R(12) * t0) * p23;
        w2 = (R(18) * t3) * p01;
        w3 = (R(4) * t2) * p01;
    } else {
        // fp32: products of (eps+beta)^2 leave the exponent range (R10): one reciprocal per weight
        R r0 = T::rcp_(b0), r1 = T::rcp_(b1), r2 = T::rcp_(b2), r3 = T::rcp_(b3);
        w0 = r0 * r0;
        w1 = (R(12) * r1) * r1;
        w2 = (R(18) * r2) * r2;
        w3 = (R(4) * r3) * r3;
    }
    R s23 = w2 + w3;
    R s123 = w1 + s23;
    den = w0 + s123;
    num12 = T::fma_(s123, R(3) * G0, T::fma_(-s23, G1, w3 * G2));
    base12 = T::fma_(R(13), D2, T::fma_(R(-10), D1, R(3) * D0));
}

// ------------------------------------------------------------------------------------------------ a-3..a-7
template <typename R>
struct SweepArgs {
    const R* U;      // stage state U_s: nf blocks of N, x fastest
    const R* P;      // pressure of U_s
    const R* W;      // scale/(E+p) of U_s
    R* L;            // right-hand side accumulator: nf blocks of N
    const R* Un;     // U^n for the stage combination (MODE 2, only read if use_un)
    R* Uout;         // next stage state (MODE 2)
    const Diag* diag;
    int slot;        // which DiagSlot holds alpha of U_s
    int nx, ny, nz, nf, nseg, use_un;
    int seg_len;     // TMA sweeps: march cells per block (multiple of 8)
    long long N;
    R eps_eff;       // 144 * weno_eps: the split fluxes are carried as 2 f^+-, beta is carried as 36 beta
    R half_inv_dx;   // 0.5 / dx
    R dt, rk_a, rk_b;
};

// MODE 0: L = -D_d;  MODE 1: L -= D_d;  MODE 2: U_next = a U^n + b (U_s + dt (L - D_d))   (Shu-Osher, R5)
// Thread = one grid line (or segment of it) of one field; lanes run over the transverse index, so for DIR = 1, 2
// a warp touches 32 consecutive x at every step of the march (coalesced); DIR = 0 lanes stride by a row.
template <typename R, int DIR, int MODE>
__global__ void __launch_bounds__(128) k_sweep(SweepArgs<R> a) {
    typedef Real<R> T;
    const int nd = DIR == 0 ? a.nx : DIR == 1 ? a.ny : a.nz;
    const long long ntrans = a.N / nd;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntrans) return;
    const int f = blockIdx.y;
    long long base, stride;
    if (DIR == 0) { base = t * a.nx; stride = 1; }
    else if (DIR == 1) { long long k = t / a.nx; base = k * (long long)a.nx * a.ny + (t - k * a.nx); stride = a.nx; }
    else { base = t; stride = (long long)a.nx * a.ny; }
    const int ls = (nd + a.nseg - 1) / a.nseg;
    const int s0 = blockIdx.z * ls;
    const int s1 = min(nd, s0 + ls);
    if (s0 >= s1) return;

    const R alpha = T::from_bits(a.diag->slot[a.slot].alpha_bits[DIR]);
    const R* __restrict__ Uf = a.U + (long long)f * a.N;
    const R* __restrict__ Ud = a.U + (long long)(1 + DIR) * a.N;
    const R* __restrict__ Wt = a.W;
    const R* __restrict__ Pp = a.P;
    const R c3 = R(39.05), eps = a.eps_eff;
    const bool is_energy = (f == 0), is_normal = (f == 1 + DIR);

    Win<R> wp, wm;
    wp.clear();
    wm.clear();
    R fp_pending = R(0);

    // split flux of cell c (index clamped = zero-gradient outflow ghosts, a-7), carried as 2 f^+- = F +- alpha U
    auto load = [&](int c, R& fp2, R& fm2) {
        c = max(0, min(nd - 1, c));
        const long long idx = base + (long long)c * stride;
        const R u = Uf[idx];
        const R md = Ud[idx];
        R F;
        if (is_energy) F = md;                                   // F^d_E = M_d
        else {
            const R vd = md * Wt[idx];
            F = u * vd;                                          // M_j v_d,  N_B v_d
            if (is_normal) F += Pp[idx];                         // + p delta_jd
        }
        fp2 = T::fma_(alpha, u, F);
        fm2 = T::fma_(-alpha, u, F);
    };

    // warm-up: cells s0-4 .. s0+3 fill both windows for the interface s0 - 1/2
    {
        R fp2, fm2;
        load(s0 - 4, fp2, fm2);
        fp_pending = fp2;
#pragma unroll
        for (int c = -3; c <= 3; ++c) {
            load(s0 + c, fp2, fm2);
            wp.push(fp_pending, c3, eps);
            wm.push(fm2, c3, eps);
            fp_pending = fp2;
        }
    }
    R* __restrict__ Lf = a.L + (long long)f * a.N;
    R fhat_prev = R(0);
    const int nsteps = s1 - s0;
#pragma unroll 6
    for (int n = 0; n <= nsteps; ++n) {
        const int i = s0 - 1 + n;                                // interface i+1/2
        if (n > 0) {
            R fp2, fm2;
            load(i + 4, fp2, fm2);
            wp.push(fp_pending, c3, eps);
            wm.push(fm2, c3, eps);
            fp_pending = fp2;
        }
        // plus side: window = cells i-3..i+3, centre i = v[0];  minus side: cells i-2..i+4 mirrored, centre i+1 = v[0]
        R bp, np_, dp, bm, nm, dm;
        weno7_side<R, false>(wp, bp, np_, dp);
        weno7_side<R, true>(wm, bm, nm, dm);
        R x;
        if (sizeof(R) == 8) x = T::fma_(np_, dm, nm * dp) * T::rcp_(dp * dm);
        else x = np_ * T::rcp_(dp) + nm * T::rcp_(dm);
        const R fhat = T::fma_((bp + bm) + x, R(1.0 / 12.0), wp.v[0] + wm.v[0]);     // = 2 F_hat_{i+1/2}
        if (n > 0) {
            const long long idx = base + (long long)i * stride;
            const R minus_div = (fhat_prev - fhat) * a.half_inv_dx;                  // -(F_hat_{i+1/2} - F_hat_{i-1/2})/dx
            if (MODE == 0) Lf[idx] = minus_div;
            else if (MODE == 1) Lf[idx] += minus_div;
            else {
                const R ltot = Lf[idx] + minus_div;
                R un = T::fma_(a.dt, ltot, Uf[idx]);
                if (a.use_un) un = T::fma_(a.rk_b, un, a.rk_a * a.Un[(long long)f * a.N + idx]);
                a.Uout[(long long)f * a.N + idx] = un;
            }
        }
        fhat_prev = fhat;
    }
}

// ------------------------------------------------------------------------------------------------ a-5: jet source
// eq. (2): the medium gains (q, q n_hat)/dx^3 in ONE cell per jet (R7); eq. (3) with T from e = g hbarc T^4 and an
// overall hbarc (R8): q = hbarc (C_R/C_F) (kappa_rad T^3 l + kappa_coll T^2) [GeV/fm], l = path length.
// The deposit cell is found with individually rounded IEEE operations (no FMA contraction) so that it is the
// same cell on any machine: idx = floor((x - x_min)/dx + 2^-20).
struct SourceArgs {
    Diag* diag;
    const JetDev* jets;
    int njets, slot, stage, commit;    // commit: add the slot's cap/NaN counts to the totals, log q, accumulate deposits
    int nx, ny, nz;
    long long N, step;
    double stage_c, dx, dt, rk_weight;
    double scale;                      // the deposit is added to `target` times this (1 for L, b dt for a stage state)
};

__device__ __forceinline__ int jet_axis_index(double x, int n, double dx) {
    const double xmin = __dmul_rn(-0.5 * (double)n, dx);
    const double a = __dadd_rn(__ddiv_rn(__dadd_rn(x, -xmin), dx), 1.0 / 1048576.0);
    const double fl = floor(a);
    if (fl < 0.0 || fl > (double)(n - 1)) return -1;
    return (int)fl;
}

template <typename R>
__global__ void k_source(SourceArgs a, const R* __restrict__ P, R* __restrict__ L /* target */) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Diag* dg = a.diag;
    const DiagSlot* s = &dg->slot[a.slot];
#pragma unroll
    for (int d = 0; d < 3; ++d) dg->alpha_last[d] = (double)Real<R>::from_bits(s->alpha_bits[d]);
    if (a.commit) {
        dg->ncap_total += s->ncap;
        dg->nan_total |= s->nan_flag;
    }
    const double HBARC = 0.1973269804;
    const double G_DOF = 47.5 * 3.14159265358979323846 * 3.14159265358979323846 / 30.0;
    const double dx3 = a.dx * a.dx * a.dx;
    for (int J = 0; J < a.njets; ++J) {
        const JetDev jt = a.jets[J];
        const double ell = __dmul_rn(__dadd_rn((double)(a.step - jt.step_added), a.stage_c), a.dt);
        const int ci = jet_axis_index(__dadd_rn(jt.x0, __dmul_rn(jt.nx, ell)), a.nx, a.dx);
        const int cj = jet_axis_index(__dadd_rn(jt.y0, __dmul_rn(jt.ny, ell)), a.ny, a.dx);
        const int ck = jet_axis_index(__dadd_rn(jt.z0, __dmul_rn(jt.nz, ell)), a.nz, a.dx);
        double q = 0.0;
        if (ci >= 0 && cj >= 0 && ck >= 0) {
            const long long c = ((long long)ck * a.ny + cj) * a.nx + ci;
            const double e_c = 3.0 * (double)P[c];
            const double T2 = sqrt(e_c / (G_DOF * HBARC));       // T^2, T in 1/fm
            const double T = sqrt(T2);
            q = HBARC * jt.crcf * (jt.k_rad * T2 * T * ell + jt.k_coll * T2);
            const double r = a.scale * (q / dx3);
            L[c] += (R)r;
            L[a.N + c] += (R)(r * jt.nx);
            L[2 * a.N + c] += (R)(r * jt.ny);
            L[3 * a.N + c] += (R)(r * jt.nz);
        }
        if (a.commit) {
            if (J < MAX_JETS) dg->last_q[a.stage][J] = q;
            const double amt = a.dt * a.rk_weight * q;
            dg->deposited[0] += amt;
            dg->deposited[1] += amt * jt.nx;
            dg->deposited[2] += amt * jt.ny;
            dg->deposited[3] += amt * jt.nz;
        }
    }
}

// ------------------------------------------------------------------------------------------------ ALU peak probe
// Register-resident FMA chains (8 independent accumulators per thread); flops = 2 * 8 * iters per thread.
template <typename R>
__global__ void __launch_bounds__(256) k_alu_peak(R* out, int iters, R x, R y) {
    R acc[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[j] = R(j) + R(threadIdx.x) * R(1e-3);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[j] = Real<R>::fma_(acc[j], x, y);
        }
    }
    R sum = R(0);
#pragma unroll
    for (int j = 0; j < 8; ++j) sum += acc[j];
    if (sum == R(123456789)) out[0] = sum;      // never true for the chosen x, y; keeps the chain alive
}

}  // namespace hydro_dev
