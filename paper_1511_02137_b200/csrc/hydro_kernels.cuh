// hydro_kernels.cuh -- device code of the hot path (sm_100a).  PRODUCT; shares nothing with oracle/.
//
// Steps of SURVEY.md 8(a) / DESIGN.md "Kernels":
//   k_prim        a-1 con2prim (p = e/3 closed form, admissibility cap R9) + a-2 wavespeeds and their global max
//   k_source      a-5 jet point source (eq. 2, 3 of the paper) + diagnostics bookkeeping
//   (the sweeps a-3, a-4, a-6, a-7 live in hydro_sweep_ring.cuh)
//
// Device layout: SoA fields of nz*ny rows with a row PITCH of nxp >= nx reals (nxp*sizeof(R) a multiple of 16 bytes,
// which TMA needs); pad columns are never read as cells.  Field stride Np = nxp*ny*nz.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace hydro_dev {

constexpr int MAX_JETS = 64;

// ------------------------------------------------------------------------------------------------ diagnostics
// One slot per "generation" of primitives (three rotate, one per stage of an RK3 step, so that every step uses the
// same sequence and one step can be replayed as a CUDA graph): k_prim fills a slot for the state it converts,
// k_source commits it to the totals when a stage actually consumes that state and clears the slot the NEXT k_prim
// will fill.
struct DiagSlot {
    unsigned long long alpha_bits[3];   // max wavespeed per direction, as the bit pattern of a non-negative real
    unsigned long long ncap;            // cells where the floor / cap of con2prim fired
    unsigned long long nan_flag;        // a non-finite conserved value was seen
    unsigned long long arg[3];          // interior linear index of a cell whose speed was (close to) the maximum: the
                                        // NEXT k_prim starts its running maxima from the exact speeds of these cells
};
constexpr int NSLOT = 3;
struct Diag {
    DiagSlot slot[NSLOT];
    long long step;                     // completed RK3 steps (device copy: jet positions of a replayed graph come from here)
    unsigned long long ncap_total;
    unsigned long long nan_total;
    unsigned long long nlim_total;      // limiter (R16): faces with theta < 1, all stages
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
    // p = e/3 = (E^2 - M^2) / (E + s) and E + p = (2E + s)/3 (from e = s - E): ONE reciprocal serves both quotients
    const R s = T::sqrt_fast(R(4) * E * E - R(3) * M2);
    const R d1 = E + s, d2 = T::fma_(R(2), E, s);
    const R r = T::rcp_fast(d1 * d2);
    p = (E * E - M2) * (r * d2);
    wt = (R(3) * sc) * (r * d1);
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
    const R* U;        // nf blocks of Np
    R* P;              // pressure
    R* W;              // wt = scale/(E+p)
    Diag* diag;
    int slot;
    int nx, nxp;       // cells per row, row pitch
    long long c0, N, Np;   // interior cells [c0, N) of this launch (a range of z planes), field stride
    long long own_lo, own_hi;   // cap events are counted for interior cells in [own_lo, own_hi) only (slab halos excluded)
    int with_alpha;    // 0: primitives only (halo planes of a z-slab: their speeds are the neighbour's business)
    int seed_slot;     // DiagSlot whose arg[] names the candidate cells (the previous stage's slot; any slot is valid)
    R e_floor, one_minus_delta;
};

// padded linear index of interior cell c (c = row*nx + i)
__device__ __forceinline__ long long pad_index(long long c, int nx, int nxp) {
    if (nx == nxp) return c;
    const long long row = c / nx;
    return row * nxp + (c - row * nx);
}

// Exact global maxima without evaluating every cell's speeds: lambda_d of a cell exceeds a threshold M iff
//     cs sqrt(rad) > M den - |v_d| (1 - cs2)   <=>   t < 0  or  rad / 3 > t^2,   t = M den - |v_d| (1 - cs2),
// which costs 3 operations instead of a square root, a reciprocal and their Newton steps.  Every thread keeps M_d = the
// largest speed it has evaluated exactly so far (times 1 - margin, so that rounding in the test can never hide a larger
// cell) and starts from the exact speeds of three candidate cells of THIS state: the cells that set the maxima of the
// previous stage's state (DiagSlot::arg) -- true cells of the launch's range, hence lower bounds of the maxima that need
// no fallback.  Smooth flow: only the warps near the fastest cells ever take the exact path.  The result is the same
// exact maximum as evaluating every cell (the candidates' owners evaluate them exactly like any other cell).
template <typename R>
__device__ __forceinline__ void cell_speeds(R Mx, R My, R Mz, R wt, R& vx, R& vy, R& vz, R& om, R& den) {
    vx = Mx * wt; vy = My * wt; vz = Mz * wt;
    const R v2 = vx * vx + vy * vy + vz * vz;
    om = R(1) - v2;
    om = om < R(0) ? R(0) : om;
    den = R(1) - v2 * R(1.0 / 3.0);
}

constexpr int PRIM_THREADS = 256;
// fp64: 2 resident blocks (126 registers, no spills; 3 blocks = 80 registers spill and measure 0.146 against 0.140 ms per
// launch at 256^3); fp32: 3 blocks.  Staging depth 2 (a third trip in flight measured the same in fp64).
#ifndef PRIM_DEPTH
#define PRIM_DEPTH 2
#endif
template <typename R>
__global__ void __launch_bounds__(PRIM_THREADS, sizeof(R) == 8 ? 2 : 3) k_prim(PrimArgs<R> a) {
    R am[3] = {R(0), R(0), R(0)};
    unsigned int ncap = 0, bad = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const R* __restrict__ U0 = a.U;
    const R* __restrict__ U1 = a.U + a.Np;
    const R* __restrict__ U2 = a.U + 2 * a.Np;
    const R* __restrict__ U3 = a.U + 3 * a.Np;
    const R margin = sizeof(R) == 8 ? R(1.0 - 1e-12) : R(1.0 - 1e-5);
    // one shared array: the staging slots of the main loop; before the loop its first reals hold the seeds, after it the
    // block reduction (static shared memory is limited to 48 KB, which three trips of staging fill)
    __shared__ __align__(16) R stg[PRIM_DEPTH][8][PRIM_THREADS];
    R* seed = &stg[0][0][0];
    if (a.with_alpha) {
        if (threadIdx.x < 3) {
            long long cs = (long long)a.diag->slot[a.seed_slot].arg[threadIdx.x];
            cs = cs < a.c0 ? a.c0 : (cs > a.N - 1 ? a.N - 1 : cs);
            const long long pc = pad_index(cs, a.nx, a.nxp);
            R p, wt, vx, vy, vz, om, den;
            int lim;
            con2prim<R>(U0[pc], U1[pc], U2[pc], U3[pc], a.e_floor, a.one_minus_delta, p, wt, lim);
            cell_speeds<R>(U1[pc], U2[pc], U3[pc], wt, vx, vy, vz, om, den);
            const R vd = threadIdx.x == 0 ? vx : threadIdx.x == 1 ? vy : vz;
            const R lam = max_wavespeed<R>(vd, den, Real<R>::rcp_fast(den), om);
            seed[threadIdx.x] = lam == lam ? lam * margin : R(0);                 // a NaN state: evaluate everything
        }
        __syncthreads();
    }
    R M[3] = {R(0), R(0), R(0)};
    long long arg[3] = {a.c0, a.c0, a.c0};
    if (a.with_alpha) {
        M[0] = seed[0]; M[1] = seed[1]; M[2] = seed[2];
        __syncthreads();                                                      // before the staging loads reuse the slots
    }
    // 1 - v_thr^2 (shrunk a little, so that rounding can only send more cells to the full test); 2 = test every cell
    auto om_threshold = [&]() {
        const R cs = R(0.57735026918962576451);
        R Mm = M[0] < M[1] ? M[0] : M[1];
        Mm = Mm < M[2] ? Mm : M[2];
        if (!(Mm > cs)) return R(2);
        const R vt = (Mm - cs) / (R(1) - Mm * cs);
        return R(1) - vt * vt * (sizeof(R) == 8 ? R(1.0 - 1e-9) : R(1.0 - 1e-4));
    };
    R om_thr = om_threshold();
    auto cell = [&](long long c0, R E, R Mx, R My, R Mz, R& p, R& wt) {
        int lim;
        con2prim<R>(E, Mx, My, Mz, a.e_floor, a.one_minus_delta, p, wt, lim);
        ncap += (c0 >= a.own_lo && c0 < a.own_hi) ? lim : 0;
        // finite check: 0 x is 0 for finite x, NaN otherwise
        const R chk = Real<R>::fma_(Mz, R(0), Real<R>::fma_(My, R(0), Real<R>::fma_(Mx, R(0), E * R(0))));
        bad |= (chk == R(0)) ? 0u : 1u;
        if (!a.with_alpha) return;
        R vx, vy, vz, om, den;
        cell_speeds<R>(Mx, My, Mz, wt, vx, vy, vz, om, den);
        // prefilter: lambda_d <= (|v| + cs) / (1 + |v| cs) in every direction (equality for v along d), so a cell with
        // |v| <= v_thr, (v_thr + cs) / (1 + v_thr cs) = min_d M_d, cannot raise any maximum: one comparison on 1 - v^2
        if (om >= om_thr) return;
        const R k23 = R(2.0 / 3.0), k13 = R(1.0 / 3.0);
        const R tx = Real<R>::fma_(M[0], den, -k23 * (vx < R(0) ? -vx : vx));
        const R ty = Real<R>::fma_(M[1], den, -k23 * (vy < R(0) ? -vy : vy));
        const R tz = Real<R>::fma_(M[2], den, -k23 * (vz < R(0) ? -vz : vz));
        const R rx = k13 * om * Real<R>::fma_(-k23 * vx, vx, den);
        const R ry = k13 * om * Real<R>::fma_(-k23 * vy, vy, den);
        const R rz = k13 * om * Real<R>::fma_(-k23 * vz, vz, den);
        const bool hot = (tx < R(0)) | (rx > tx * tx) | (ty < R(0)) | (ry > ty * ty) | (tz < R(0)) | (rz > tz * tz);
        if (hot) {                                                   // rare: this cell may raise a maximum
            const R inv_den = Real<R>::rcp_fast(den);
            const R lx = max_wavespeed<R>(vx, den, inv_den, om);
            const R ly = max_wavespeed<R>(vy, den, inv_den, om);
            const R lz = max_wavespeed<R>(vz, den, inv_den, om);
            if (lx > am[0]) { am[0] = lx; arg[0] = c0; }
            if (ly > am[1]) { am[1] = ly; arg[1] = c0; }
            if (lz > am[2]) { am[2] = lz; arg[2] = c0; }
            const R mx = lx * margin, my = ly * margin, mz = lz * margin;
            M[0] = mx > M[0] ? mx : M[0];
            M[1] = my > M[1] ? my : M[1];
            M[2] = mz > M[2] ? mz : M[2];
            om_thr = om_threshold();
        }
    };
    // two cells per trip, staged through thread-private shared-memory slots with cp.async, two trips deep: the loads of the
    // next trip are in flight while this trip's arithmetic runs and cost no registers (ncu of the plain loop: 40 % of the
    // issue cycles on the long scoreboard at 24 warps/SM; register double-buffering at 5 x 128 threads was slower still)
    if (a.nx == a.nxp && !(a.c0 & 1) && !(a.N & 1)) {
        // dense rows (the usual case): the two cells of a trip are NEIGHBOURS, moved as one 2-real vector per field
        // (16-byte cp.async / shared-memory loads / stores in fp64): half the memory instructions, 512-byte warp accesses
        struct __align__(2 * sizeof(R)) R2 { R x, y; };
        R2(*sv)[4][PRIM_THREADS] = reinterpret_cast<R2(*)[4][PRIM_THREADS]>(&stg[0][0][0]);
        const long long Q = a.N >> 1;
        auto fetchv = [&](int buf, long long q) {
            const R* src[4] = {U0 + 2 * q, U1 + 2 * q, U2 + 2 * q, U3 + 2 * q};
#pragma unroll
            for (int v = 0; v < 4; ++v) {
                const unsigned dst = (unsigned)__cvta_generic_to_shared(&sv[buf][v][threadIdx.x]);
                if (sizeof(R) == 8) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src[v]) : "memory");
                else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src[v]) : "memory");
            }
        };
        long long q = (a.c0 >> 1) + (long long)blockIdx.x * blockDim.x + threadIdx.x;
        int buf = 0;
#pragma unroll
        for (int d = 0; d < PRIM_DEPTH - 1; ++d) {                            // PRIM_DEPTH - 1 trips in flight
            if (q + d * stride < Q) fetchv(d, q + d * stride);
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        for (; q < Q; q += stride, buf = buf + 1 == PRIM_DEPTH ? 0 : buf + 1) {
            const int bn = buf == 0 ? PRIM_DEPTH - 1 : buf - 1;               // the slot the previous trip has just freed
            if (q + (PRIM_DEPTH - 1) * stride < Q) fetchv(bn, q + (PRIM_DEPTH - 1) * stride);
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group %0;" ::"n"(PRIM_DEPTH - 1) : "memory");   // this trip's four vectors have landed
            const R2 E = sv[buf][0][threadIdx.x], Mx = sv[buf][1][threadIdx.x], My = sv[buf][2][threadIdx.x],
                     Mz = sv[buf][3][threadIdx.x];
            R2 p, w;
            cell(2 * q, E.x, Mx.x, My.x, Mz.x, p.x, w.x);
            cell(2 * q + 1, E.y, Mx.y, My.y, Mz.y, p.y, w.y);
            *reinterpret_cast<R2*>(a.P + 2 * q) = p;
            *reinterpret_cast<R2*>(a.W + 2 * q) = w;
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    } else {
        auto fetch = [&](int buf, long long cc) {
            const long long q1 = pad_index(cc, a.nx, a.nxp), q2 = pad_index(cc + stride, a.nx, a.nxp);
            const R* src[8] = {U0 + q1, U1 + q1, U2 + q1, U3 + q1, U0 + q2, U1 + q2, U2 + q2, U3 + q2};
#pragma unroll
            for (int v = 0; v < 8; ++v) {
                const unsigned dst = (unsigned)__cvta_generic_to_shared(&stg[buf][v][threadIdx.x]);
                if (sizeof(R) == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src[v]) : "memory");
                else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src[v]) : "memory");
            }
        };
        long long c = a.c0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
        int buf = 0;
        if (c + stride < a.N) fetch(0, c);
        asm volatile("cp.async.commit_group;" ::: "memory");
        for (; c + stride < a.N; c += 2 * stride, buf ^= 1) {
            const long long cn = c + 2 * stride;
            if (cn + stride < a.N) fetch(buf ^ 1, cn);
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 1;" ::: "memory");              // this trip's eight values have landed
            const R E = stg[buf][0][threadIdx.x], Mx = stg[buf][1][threadIdx.x], My = stg[buf][2][threadIdx.x],
                    Mz = stg[buf][3][threadIdx.x];
            const R E2 = stg[buf][4][threadIdx.x], Mx2 = stg[buf][5][threadIdx.x], My2 = stg[buf][6][threadIdx.x],
                    Mz2 = stg[buf][7][threadIdx.x];
            const long long p1 = pad_index(c, a.nx, a.nxp), p2 = pad_index(c + stride, a.nx, a.nxp);
            R p, w;
            cell(c, E, Mx, My, Mz, p, w);
            a.P[p1] = p; a.W[p1] = w;
            cell(c + stride, E2, Mx2, My2, Mz2, p, w);
            a.P[p2] = p; a.W[p2] = w;
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        if (c < a.N) {
            const long long p1 = pad_index(c, a.nx, a.nxp);
            R p, w;
            cell(c, U0[p1], U1[p1], U2[p1], U3[p1], p, w);
            a.P[p1] = p; a.W[p1] = w;
        }
    }
    // warp reduction by shuffles, then one atomic per block on the bit pattern (non-negative reals order like
    // unsigned integers; the max is exact, hence order independent)
    unsigned long long ab[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) ab[d] = Real<R>::to_bits(am[d]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const unsigned long long o = __shfl_xor_sync(0xffffffffu, ab[d], off);
            const long long oa = __shfl_xor_sync(0xffffffffu, arg[d], off);
            if (o > ab[d]) { ab[d] = o; arg[d] = oa; }
        }
        ncap += __shfl_xor_sync(0xffffffffu, ncap, off);
        bad |= __shfl_xor_sync(0xffffffffu, bad, off);
    }
    __syncthreads();                                                          // every thread is done with its staging slots
    unsigned long long(*sm)[8] = reinterpret_cast<unsigned long long(*)[8]>(&stg[0][0][0]);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) {
        sm[warp][0] = ab[0]; sm[warp][1] = ab[1]; sm[warp][2] = ab[2]; sm[warp][3] = ncap; sm[warp][4] = bad;
        sm[warp][5] = (unsigned long long)arg[0]; sm[warp][6] = (unsigned long long)arg[1]; sm[warp][7] = (unsigned long long)arg[2];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long r[5] = {0, 0, 0, 0, 0}, ra[3] = {0, 0, 0};
        const int nw = blockDim.x >> 5;
        for (int w = 0; w < nw; ++w) {
            for (int d = 0; d < 3; ++d) if (sm[w][d] > r[d]) { r[d] = sm[w][d]; ra[d] = sm[w][5 + d]; }
            r[3] += sm[w][3];
            r[4] |= sm[w][4];
        }
        DiagSlot* s = &a.diag->slot[a.slot];
        if (a.with_alpha)
            for (int d = 0; d < 3; ++d)
                if (r[d] && atomicMax(&s->alpha_bits[d], r[d]) < r[d]) s->arg[d] = ra[d];   // the last raiser holds the maximum
        if (r[3]) atomicAdd(&s->ncap, r[3]);
        if (r[4]) atomicOr(&s->nan_flag, 1ull);
    }
}

// primitives for hydro_get_fields(which = 1): (e, vx, vy, vz [, n]); `out` has the same pitched layout as U
template <typename R>
__global__ void __launch_bounds__(256) k_prims_out(const R* __restrict__ U, R* __restrict__ out, long long N, long long Np,
                                                   int nx, int nxp, int nf, R e_floor, R one_minus_delta) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long c0 = (long long)blockIdx.x * blockDim.x + threadIdx.x; c0 < N; c0 += stride) {
        const long long c = pad_index(c0, nx, nxp);
        R E = U[c], Mx = U[Np + c], My = U[2 * Np + c], Mz = U[3 * Np + c];
        R p, wt;
        int lim;
        con2prim<R>(E, Mx, My, Mz, e_floor, one_minus_delta, p, wt, lim);
        R vx = Mx * wt, vy = My * wt, vz = Mz * wt;
        out[c] = R(3) * p;
        out[Np + c] = vx;
        out[2 * Np + c] = vy;
        out[3 * Np + c] = vz;
        if (nf > 4) {
            R om = R(1) - (vx * vx + vy * vy + vz * vz);
            om = om < R(0) ? R(0) : om;
            out[4 * Np + c] = U[4 * Np + c] * Real<R>::sqrt_(om);
        }
    }
}

// ------------------------------------------------------------------------------------------------ limiter: U^L (R16, f-1)
// First-order Lax-Friedrichs update  U^L = U - (dt/dx) sum_d (F^L_{i+1/2} - F^L_{i-1/2}),
// F^L_{i+1/2} = [(F_i + alpha U_i) + (F_{i+1} - alpha U_{i+1})] / 2, neighbours clamped (zero-gradient ghosts).
template <typename R>
struct LowArgs {
    const R* U; const R* P; const R* W; R* UL;
    const Diag* diag;
    int slot, nx, ny, nz, nxp, nf;
    long long N, Np;
    R lam;                       // dt / dx
};

// one cell's inputs of the first-order update (the kernel is k_lowup_tma, hydro_lowup.cuh)
template <typename R, int NF>
struct LowCell { R u[NF], w, p; };

// (F^d_q - s alpha U_q) of a cell, s = +1 (upper neighbour) or -1 (lower neighbour)
template <typename R, int NF>
__device__ __forceinline__ R low_term(const LowCell<R, NF>& x, int d, int q, R s_alpha) {
    R F;
    if (q == 0) F = x.u[1 + d];
    else {
        F = x.u[q] * (x.u[1 + d] * x.w);
        if (q == 1 + d) F += x.p;
    }
    return F - s_alpha * x.u[q];
}

// out = (A - B) / dt over the interior cells: L of the limited scheme for hydro_eval_rhs, from the limited Euler update
template <typename R>
__global__ void __launch_bounds__(256) k_diff(const R* __restrict__ A, const R* __restrict__ B, R* __restrict__ out, long long n, R inv_dt) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += stride) out[c] = (A[c] - B[c]) * inv_dt;
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
    int zero_slot;                     // >= 0: clear this DiagSlot (the one the next k_prim fills)
    int advance;                       // 1: this is the last stage of a step: diag->step += 1 afterwards
    int nx, ny, nz, nxp;
    int nz_global, k_offset, own_lo, own_hi;   // z-slab (f-4): global planes, global index of local plane 0, owned local planes
    long long N /* field stride Np */;
    double stage_c, dx, dt, rk_weight;
    double scale;                      // the deposit is added to `target` times this (1 for L, b dt for a stage state)
    double sigma;                      // Gaussian deposit width [fm] (R15); 0 = point deposit (R7)
};

__device__ __forceinline__ int jet_axis_index(double x, int n, double dx) {
    const double xmin = __dmul_rn(-0.5 * (double)n, dx);
    const double a = __dadd_rn(__ddiv_rn(__dadd_rn(x, -xmin), dx), 1.0 / 1048576.0);
    const double fl = floor(a);
    if (fl < 0.0 || fl > (double)(n - 1)) return -1;
    return (int)fl;
}

constexpr int SOURCE_THREADS = 256;

// One block.  Thread 0 does the bookkeeping and the point deposit (R7); with sigma > 0 (reading R15)
// the whole block spreads q over the (2R+1)^3 cells around the R7 cell with normalised Gaussian weights
// w = exp(-(r^2 - r0^2) / (2 sigma^2)) (r: cell centre to jet position, r0: that of the R7 cell), R = ceil(3 sigma/dx -
// 2^-20) in [1, 8]; the sum of the weights is reduced in a fixed order (bitwise reproducible); the part of the cube
// outside the grid is lost.  Jets are processed one after the other, so overlapping deposits add in a fixed order.
template <typename R>
__global__ void __launch_bounds__(SOURCE_THREADS) k_source(SourceArgs a, const R* __restrict__ P, R* __restrict__ L /* target */) {
    __shared__ double sh_q, sh_pos[3], sh_red[SOURCE_THREADS];
    __shared__ int sh_c[3];
    const int tid = threadIdx.x;
    Diag* dg = a.diag;
    const long long step = dg->step;                                 // read by every thread before thread 0 advances it
    __syncthreads();
    if (tid == 0) {
        if (a.zero_slot >= 0) {
            DiagSlot* z = &dg->slot[a.zero_slot];
            z->alpha_bits[0] = z->alpha_bits[1] = z->alpha_bits[2] = 0ull;
            z->ncap = 0ull;
            z->nan_flag = 0ull;
        }
        if (a.advance) dg->step = step + 1;
        const DiagSlot* s = &dg->slot[a.slot];
#pragma unroll
        for (int d = 0; d < 3; ++d) dg->alpha_last[d] = (double)Real<R>::from_bits(s->alpha_bits[d]);
        if (a.commit) {
            dg->ncap_total += s->ncap;
            dg->nan_total |= s->nan_flag;
        }
    }
    const double HBARC = 0.1973269804;
    const double G_DOF = 47.5 * 3.14159265358979323846 * 3.14159265358979323846 / 30.0;
    const double dx3 = a.dx * a.dx * a.dx;
    for (int J = 0; J < a.njets; ++J) {
        const JetDev jt = a.jets[J];
        if (tid == 0) {
            const double ell = __dmul_rn(__dadd_rn((double)(step - jt.step_added), a.stage_c), a.dt);
            const double xj = __dadd_rn(jt.x0, __dmul_rn(jt.nx, ell)), yj = __dadd_rn(jt.y0, __dmul_rn(jt.ny, ell)),
                         zj = __dadd_rn(jt.z0, __dmul_rn(jt.nz, ell));
            const int ci = jet_axis_index(xj, a.nx, a.dx);
            const int cj = jet_axis_index(yj, a.ny, a.dx);
            int ck = jet_axis_index(zj, a.nz_global, a.dx);
            if (ck >= 0) { ck -= a.k_offset; if (ck >= a.nz) ck = -1; }        // global -> local plane; outside the local array: no deposit here
            const bool owned = ck >= a.own_lo && ck < a.own_hi;
            double q = 0.0;
            // a point deposit into a halo plane would be overwritten by the next exchange: skipped (its P may be stale)
            if (ci >= 0 && cj >= 0 && ck >= 0 && (owned || a.sigma > 0.0)) {
                const long long c = ((long long)ck * a.ny + cj) * a.nxp + ci;
                const double e_c = 3.0 * (double)P[c];
                const double T2 = sqrt(e_c / (G_DOF * HBARC));       // T^2, T in 1/fm
                const double T = sqrt(T2);
                q = HBARC * jt.crcf * (jt.k_rad * T2 * T * ell + jt.k_coll * T2);
                if (!(a.sigma > 0.0)) {
                    const double r = a.scale * (q / dx3);
                    L[c] += (R)r;
                    L[a.N + c] += (R)(r * jt.nx);
                    L[2 * a.N + c] += (R)(r * jt.ny);
                    L[3 * a.N + c] += (R)(r * jt.nz);
                }
            }
            if (a.commit) {
                if (J < MAX_JETS) dg->last_q[a.stage][J] = owned ? q : 0.0;
                const double amt = owned ? a.dt * a.rk_weight * q : 0.0;
                dg->deposited[0] += amt;
                dg->deposited[1] += amt * jt.nx;
                dg->deposited[2] += amt * jt.ny;
                dg->deposited[3] += amt * jt.nz;
            }
            sh_q = q; sh_pos[0] = xj; sh_pos[1] = yj; sh_pos[2] = zj;
            sh_c[0] = ci; sh_c[1] = cj; sh_c[2] = ck;
        }
        if (!(a.sigma > 0.0)) continue;                              // uniform: no barrier needed for the point deposit
        __syncthreads();
        const int ci = sh_c[0], cj = sh_c[1], ck = sh_c[2];
        const double q = sh_q;
        if (ci >= 0 && cj >= 0 && ck >= 0) {                         // uniform across the block
            int Rr = (int)ceil(__dadd_rn(__ddiv_rn(__dmul_rn(3.0, a.sigma), a.dx), -1.0 / 1048576.0));
            Rr = Rr < 1 ? 1 : (Rr > 8 ? 8 : Rr);
            const int side = 2 * Rr + 1, ncell = side * side * side;
            const double inv2s2 = 1.0 / (2.0 * a.sigma * a.sigma);
            const double x0c = ((ci + 0.5) - 0.5 * a.nx) * a.dx - sh_pos[0], y0c = ((cj + 0.5) - 0.5 * a.ny) * a.dx - sh_pos[1],
                         z0c = ((ck + a.k_offset + 0.5) - 0.5 * a.nz_global) * a.dx - sh_pos[2];
            const double r02 = x0c * x0c + y0c * y0c + z0c * z0c;
            auto weight = [&](int s, int& i2, int& j2, int& k2) {
                const int di = s % side - Rr, dj = (s / side) % side - Rr, dk = s / (side * side) - Rr;
                i2 = ci + di; j2 = cj + dj; k2 = ck + dk;
                const double ddx = ((i2 + 0.5) - 0.5 * a.nx) * a.dx - sh_pos[0];
                const double ddy = ((j2 + 0.5) - 0.5 * a.ny) * a.dx - sh_pos[1];
                const double ddz = ((k2 + a.k_offset + 0.5) - 0.5 * a.nz_global) * a.dx - sh_pos[2];
                return exp(-((ddx * ddx + ddy * ddy + ddz * ddz) - r02) * inv2s2);
            };
            double part = 0.0;
            int i2, j2, k2;
            for (int s = tid; s < ncell; s += SOURCE_THREADS) part += weight(s, i2, j2, k2);
            sh_red[tid] = part;
            __syncthreads();
            for (int off = SOURCE_THREADS / 2; off > 0; off >>= 1) {
                if (tid < off) sh_red[tid] += sh_red[tid + off];
                __syncthreads();
            }
            const double norm = a.scale * q / (sh_red[0] * dx3);
            for (int s = tid; s < ncell; s += SOURCE_THREADS) {
                const double w = weight(s, i2, j2, k2);
                if (i2 < 0 || i2 >= a.nx || j2 < 0 || j2 >= a.ny || k2 < 0 || k2 >= a.nz) continue;
                const long long c = ((long long)k2 * a.ny + j2) * a.nxp + i2;
                const double r = norm * w;
                L[c] += (R)r;
                L[a.N + c] += (R)(r * jt.nx);
                L[2 * a.N + c] += (R)(r * jt.ny);
                L[3 * a.N + c] += (R)(r * jt.nz);
            }
        }
        __syncthreads();                                             // the next jet may touch the same cells / shared slots
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
