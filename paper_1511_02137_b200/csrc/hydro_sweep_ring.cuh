// hydro_sweep_ring.cuh -- the WENO7-LF sweep kernels of the hot path (sm_100a, fp64).  PRODUCT.
//
// Steps a-3 (WENO7 reconstruction of the Lax-Friedrichs split fluxes), a-4 (flux divergence,
// eq. 1), a-6 (SSP-RK3 stage combination) and a-7 (outflow ghosts) of SURVEY.md 8(a), organised
// around the one resource that bounds them, the FP64 pipe:
//
//   block   = 32 lanes x NF field-warps (NF = 1: the single warp of the baryon-density kernel, see BARYON below).
//             The lanes are 32 neighbouring grid lines (consecutive x for the y/z
//             sweeps, consecutive y for the x sweep); warp f reconstructs conserved field f, so the warps of a
//             block share every input row: U (all fields), W = scale/(E+p) and P.
//   input   = a ring of 2 or 3 (ring_nstage) shared-memory stages, each CH = 8 march cells x 32 lanes of (U[NF], W, P),
//             filled by one thread with cp.async.bulk.tensor (TMA) box loads that complete on an mbarrier, one
//             chunk ahead of the arithmetic.  The x sweep uses the 64-byte TMA swizzle so that lane = row reads
//             its own row with a 2-way bank conflict at most.
//   window  = every thread marches along the sweep axis and keeps, per split sign, the undivided differences of
//             the last cells in ROTATING registers: slot = march cell mod 8, all indices compile-time constants
//             in a fully unrolled 8-row chunk body, so the window never moves through registers and the body has
//             no branches (r1_b profile: 45-50 % of the issued instructions of the previous kernel were moves).
//   ghosts  = TMA zero-fills out-of-range cells; in the (at most two) chunks of a line that hold ghost rows the
//             zero rows are overwritten in shared memory with the edge cell's row (zero-gradient outflow, R8b).
//   output  = a shared-memory tile per chunk, written back with ONE TMA op per chunk:
//               OUT_STORE     L        = c (F_{i-1/2} - F_{i+1/2})                    tensor store
//               OUT_REDUCE    target  += c (F_{i-1/2} - F_{i+1/2})                    tensor reduce-add (in L2)
//               OUT_COMBINE1  U_next   = U_s + dt L_x                                 tensor store   (stage 1)
//               OUT_COMBINE   U_next   = a U^n + b (U_s + dt L_x)                     tensor store   (stages 2, 3)
//             The stage update is linear in L = L_x + L_y + L_z + S, so the x sweep writes the combined state with
//             its own part and the y and z sweeps (and the source kernel) add b dt L_y, b dt L_z (b dt S) to it.
//             No thread ever waits on a global load or store; out-of-range rows and lanes are clipped by TMA.
#pragma once
#include <cuda.h>
#include "hydro_kernels.cuh"

namespace hydro_dev {

constexpr int RING_CH = 8;                 // march cells per chunk
constexpr int RING_NSTAGE_MAX = 3;
constexpr int RING_SUB = RING_CH * 32;     // reals per sub-tile (one field, one chunk)

enum { OUT_STORE = 0, OUT_REDUCE = 1, OUT_COMBINE1 = 2, OUT_COMBINE = 3 };
// input ring depth: chunk m (current) and m+1 (in flight); the combine kernels also read U_s of chunk m-1's last rows (their
// output cells lag the march by 4) -- unless the limiter's U^L tiles replace U_s there
__host__ __device__ constexpr int ring_nstage(int out, int lim) {
    return ((out == OUT_COMBINE1 || out == OUT_COMBINE) && !lim) ? 3 : 2;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Bounded wait: a TMA load that never completes (bad tensor map) must become a CUDA error, not a hung GPU.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    const uint32_t addr = smem_u32(bar);
    for (unsigned spin = 0; spin < (1u << 22); ++spin) {
        uint32_t done;
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(addr), "r"(parity)
            : "memory");
        if (done) return;
    }
    __trap();
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2,
                                            int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ void tma_store_4d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];" ::"l"(tm),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
                 : "memory");
}
__device__ __forceinline__ void tma_reduce_add_4d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2,
                                                  int c3) {
    asm volatile("cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4, %5}], [%1];" ::"l"(tm),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
                 : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// shared-memory plan of one launch (host and device agree through these functions); units: reals
__host__ __device__ constexpr int ring_stage_reals(int nf, int lim = 0) { return (lim ? nf + 2 : nf + 2) * RING_SUB; }
__host__ __device__ constexpr int ring_smem_bytes(int nf, int out, int esz, int lim = 0) {
    return (ring_nstage(out, lim) * ring_stage_reals(nf, lim)   // input ring
            + (lim ? (2 * nf + 1) * RING_SUB : 0)          // limiter: two U^L tiles (this chunk, previous chunk) + theta tile
            + 2 * nf * RING_SUB                            // two output tiles
            + (out == OUT_COMBINE ? (lim ? 1 : 2) * nf * RING_SUB : 0)   // U^n tiles: two riding with the input stages; limiter: one
            + RING_SUB) * esz                              // one tile of zeros
           + 64;                                           // mbarriers
}
// limiter x sweeps: 16-byte row-pair accesses of the swizzled tiles (conflict-free) in 1: phase B (theta), 2: + phase C (emit),
// 3: + phase A (corrections); 0: 8-byte accesses everywhere (A/B knob; measured 2.03 / 1.96 / 1.84 / 1.83 ms per step for 0..3)
#ifndef RING_LIM_X_PAIRS
#define RING_LIM_X_PAIRS 3
#endif
#ifndef RING_F64_BLOCKS
#define RING_F64_BLOCKS 3
#endif
#ifndef RING_F32_BLOCKS
#define RING_F32_BLOCKS 6
#endif
// resident blocks per SM the kernels are compiled for (registers: 65536 / (32 NF threads x blocks))
__host__ __device__ constexpr int ring_blocks_per_sm(int nf, int esz, int out = OUT_COMBINE, int lim = 0) {
    if (nf == 1) return 8;                                    // baryon kernel: one warp, 24-28 KB of shared memory
    if (lim) return nf == 4 ? 3 : 2;                          // <= 68 KB and <= 168 registers; 5 warps: 2
    // nf = 5 in fp64: 3 blocks (<= 136 registers, 64 KB) except the combine kernel with its U^n tiles (84 KB): 2
    return esz == 8 ? (nf == 4 ? RING_F64_BLOCKS : (out != OUT_COMBINE ? 3 : 2)) : (nf == 4 ? RING_F32_BLOCKS : 4);
}

struct RingMaps {
    CUtensorMap U, W, P;       // loads: stage state (NF fields per box), W and P (one field per box)
                               // NF = 1 (baryon kernel): U, Un, Out are one-field-box maps of the 5-field buffers, P is unused
    CUtensorMap Un;            // load : U^n at the output cells (OUT_COMBINE)
    CUtensorMap Out;           // store / reduce target (NF fields per box)
    CUtensorMap UL;            // load : first-order update U^L (limiter, R16)
};

struct RingArgs {
    const Diag* diag;
    int slot;                  // which DiagSlot holds alpha of U_s
    int nx, ny, nz;
    int seg_len;               // march cells per block (multiple of RING_CH)
    int n_long, short_nseg, short_len;   // tail-split mode (n_long >= 0), see the kernel
    double eps_eff;            // WENO7: 144 * weno_eps / 39 (the split fluxes are carried as 2 f^+-, beta as 36 beta / 39); WENO5: 48 * weno_eps
    double coef;               // OUT_STORE / OUT_REDUCE: c = [b dt] / (2 dx);  OUT_COMBINE*: 1 / (2 dx)
    double dt, rk_a, rk_b;
    double k3lam;              // limiter: 6 dt/dx times the correction C = corr / (2 KW) (the exchange tile holds corr = KW x 2 C)
    unsigned long long* nlim;  // limiter: count of faces with theta < 1
    int own_lo, own_hi;        // limiter count: only faces of owned planes (z sweep: faces whose LOWER cell is owned, and the
                               // physical boundary face below plane 0), so that sums over ranks are global figures
};

// element offset inside a sub-tile of march row r (0..7) for this lane
template <int DIR, typename R>
__device__ __forceinline__ int sub_off(int r, int lane) {
    if (DIR == 0) {
        // dense box layout (8 cells of x fastest, 32 rows of y):
        //   fp64: byte = lane*64 + r*8, TMA 64-byte swizzle: 16-byte chunk index (bits 4..5) ^= address bits 7..8
        //   fp32: byte = lane*32 + r*4, TMA 32-byte swizzle: 16-byte chunk index (bit 4)     ^= address bit 7
        if (sizeof(R) == 8) return lane * 8 + ((((r >> 1) ^ ((lane >> 1) & 3)) << 1) | (r & 1));
        return lane * 8 + ((((r >> 2) ^ ((lane >> 2) & 1)) << 2) | (r & 3));
    }
    return r * 32 + lane;
}

// ------------------------------------------------------------------------------------------------ rotating window
// Undivided differences of one split flux along the march, slot = march row mod 8:
//   V = value, D = V - V_prev, E = D - D_prev, T = E - E_prev, G = T - T_prev, S = cT T^2 + eps.
// Live at any time (WENO7): 4 V, 6 D, 5 E, 4 S, 3 G, 1 T (the other slots are dead registers).
// The kernels are issue-bound with every FP64 instruction taking two issue cycles, so the scalings are chosen
// to leave no multiplication by a constant that an FMA coefficient can absorb:
//   WENO7: all differences are carried UNSCALED (the push is four subtractions + S); the smoothness indicators are carried
//          divided by 39, beta' = (lam/sqrt(39))^2 + m^2 + (39.05/39) T^2 + eps/39 -- lam is a linear form of the D's whose
//          coefficients take the 1/sqrt(39), the m's enter as plain squares; the weights only see ratios of the betas.
//   WENO5: the split fluxes are carried times sV = sqrt(3) (one multiplication per row), so l' = sqrt(3) l enters
//          12 beta = 13 E^2 + 3 l^2 as a plain square; E is carried times sqrt(13) in all (one multiplication per push, factor
//          sE = sqrt(13/3) on top of sV), the G slots hold T = E - E_prev (the candidates' differences).
template <int ORDER> struct WinScale;
template <> struct WinScale<7> {
    static constexpr double sE = 6.2449979983983982058, iE = 0.16012815380508713318;      // sqrt(39), 1/sqrt(39)
    static constexpr double cT = 39.05 / 39.0;                                            // (39.05 T^2) / 39
    static constexpr double sV = 1.0;
};
template <> struct WinScale<5> {
    static constexpr double sV = 1.7320508075688772935, iV = 0.57735026918962576451;      // sqrt(3), 1/sqrt(3)
    static constexpr double sE = 2.0816659994661327353;                                   // sqrt(13/3): E carried = sqrt(13) E
    static constexpr double iE = 0.27735009811261456101;                                  // 1/sqrt(13)
};
template <typename R>
struct RotWin {
    R V[8], D[8], E[8], S[8], G[8], T;
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int j = 0; j < 8; ++j) { V[j] = R(0); D[j] = R(0); E[j] = R(0); S[j] = R(0); G[j] = R(0); }
        T = R(0);
    }
};

template <int r, int ORDER, typename R>
__device__ __forceinline__ void rot_push(RotWin<R>& w, R x, R eps) {
    constexpr int p = (r + 7) & 7;
    const R dn = x - w.V[p];
    if (ORDER == 7) {
        const R en = dn - w.D[p];
        const R tn = en - w.E[p];
        w.G[r] = tn - w.T;
        w.S[r] = Real<R>::fma_(R(WinScale<7>::cT) * tn, tn, eps);
        w.T = tn;
        w.E[r] = en;
    } else {
        const R en = R(WinScale<5>::sE) * (dn - w.D[p]);
        w.G[r] = en - w.E[p];                                 // T of the WENO5 window
        w.E[r] = en;
    }
    w.V[r] = x;
    w.D[r] = dn;
}

// reciprocal of a normal, well-scaled double: hardware seed (the upper 32 bits of the operand and of the result,
// i.e. a relative error e of about 2^-20) + one cubic step r (1 + e + e^2), error e^3 ~ 2^-60
__device__ __forceinline__ double rcp_cubic(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double e = fma(-x, r, 1.0);
    const double t = fma(e, e, e);
    return fma(r, t, r);
}
__device__ __forceinline__ float rcp_ulp(float x) {      // MUFU.RCP: 1 ulp, enough for the fp32 variant (R10)
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// One WENO7-JS reconstruction (r = 4) from the 1st..4th undivided differences in stencil order (D_j, E_j, G_j unscaled)
// and S_j = (39.05 T_j^2 + eps) / 39 (formulas: DESIGN.md "WENO7 in difference form"):
//   candidates   12 (q_0 - x_c) = 3 D_0 - 10 D_1 + 13 D_2,  12 (q_1-q_0) = 3 G_0,  12 (q_2-q_1) = -G_1,  12 (q_3-q_2) = G_2
//   smoothness   (36 beta_k + eps) / 39 = Lam_k^2 + m_k^2 + S_k,   Lam_k = lam_k / sqrt(39),
//                lam_0 = 2 D_0 - 7 D_1 + 11 D_2, lam_1 = lam_0 + 2 G_0, lam_2 = lam_1 - G_1, lam_3 = lam_2 + 2 G_2,
//                m_0 = 2 E_1 - E_0,  m_1 = m_2 = E_2,  m_3 = 2 E_3 - E_4
//   weights      fp64: omega_k ~ d_k prod_{j != k} (eps + beta_j)^2,  d = (1, 12, 18, 4)/35  (common denominator;
//                range-safe in fp64);  fp32: omega_k ~ d_k (1/(eps + beta_k))^2, one reciprocal each (R10);
//                the d_k are applied as (1/4, 3, 4.5, 1): a common factor drops out of num/den
// Returns base12 = 12 (q_0 - x_c) and num12/den = 12 sum_k omega_k (q_k - q_0):  W = x_c + (base12 + num12/den)/12.
template <typename R>
__device__ __forceinline__ void weno7_diff(R D0, R D1, R D2, R E0, R E1, R E2, R E3, R E4, R S0, R S1, R S2, R S3,
                                           R G0, R G1, R G2, R& base12, R& num12, R& den) {
    typedef Real<R> T;
    constexpr double iE = WinScale<7>::iE;
    const R lam0 = T::fma_(R(11 * iE), D2, T::fma_(R(-7 * iE), D1, R(2 * iE) * D0));
    const R lam1 = T::fma_(R(2 * iE), G0, lam0);
    const R lam2 = T::fma_(R(-iE), G1, lam1);
    const R lam3 = T::fma_(R(2 * iE), G2, lam2);
    const R m0 = T::fma_(R(2), E1, -E0);
    const R m3 = T::fma_(R(2), E3, -E4);
    const R b0 = T::fma_(lam0, lam0, T::fma_(m0, m0, S0));
    const R b1 = T::fma_(lam1, lam1, T::fma_(E2, E2, S1));
    const R b2 = T::fma_(lam2, lam2, T::fma_(E2, E2, S2));
    const R b3 = T::fma_(lam3, lam3, T::fma_(m3, m3, S3));
    R u0, u1, u2, u3;
    if (sizeof(R) == 8) {
        const R t0 = b0 * b0, t1 = b1 * b1, t2 = b2 * b2, t3 = b3 * b3;
        const R p01 = t0 * t1, p23 = t2 * t3;
        u0 = t1 * p23; u1 = t0 * p23; u2 = t3 * p01; u3 = t2 * p01;
    } else {
        const float r0 = rcp_ulp((float)b0), r1 = rcp_ulp((float)b1), r2 = rcp_ulp((float)b2), r3 = rcp_ulp((float)b3);
        u0 = r0 * r0; u1 = r1 * r1; u2 = r2 * r2; u3 = r3 * r3;
    }
    const R a23 = T::fma_(R(4.5), u2, u3);
    const R a123 = T::fma_(R(3), u1, a23);
    den = T::fma_(R(0.25), u0, a123);
    num12 = T::fma_(a123, R(3) * G0, T::fma_(-a23, G1, u3 * G2));
    base12 = T::fma_(R(WinScale<7>::sE), lam0, m0);       // 3 D_0 - 10 D_1 + 13 D_2 = lam_0 + m_0 identically
}

// One WENO5-JS reconstruction (r = 3) from the differences of the stencil values
// x_0..x_4 (centre x_2), D_j = x_{j+1} - x_j, E_j = D_{j+1} - D_j.  Carried (RotWin): D' = sqrt(3) D, E' = sqrt(13) E,
// Ta = E'_1 - E'_0, Tb = E'_2 - E'_1:
//   candidates   6 (q_0 - x_2) = 5 D_1 - 2 D_0,   6 (q_1 - q_0) = 2 (E_1 - E_0),   6 (q_2 - q_1) = -(E_2 - E_1)
//   smoothness   12 beta_k + eps = E'_k^2 + l'_k^2 + eps,  l'_0 = 3 D'_1 - D'_0,  l'_1 = D'_1 + D'_2,  l'_2 = 3 D'_2 - D'_3
//   weights      omega_k ~ d_k / (eps + beta_k)^2,  d = (1, 6, 3)/10 applied as (1/3, 2, 1)  (fp64: common denominator;
//                fp32: reciprocals)
// Returns base6 = 6 (q_0 - x_2) and num6s/den = sqrt(13) 6 sum_k omega_k (q_k - q_0):  W = x_2 + (base6 + num6s/(sqrt(13) den))/6.
template <typename R>
__device__ __forceinline__ void weno5_diff(R D0, R D1, R D2, R D3, R E0, R E1, R E2, R Ta, R Tb, R eps, R& base6, R& num6s,
                                           R& den) {
    typedef Real<R> T;
    const R l0 = T::fma_(R(3), D1, -D0);
    const R l1 = D1 + D2;
    const R l2 = T::fma_(R(3), D2, -D3);
    const R b0 = T::fma_(E0, E0, T::fma_(l0, l0, eps));
    const R b1 = T::fma_(E1, E1, T::fma_(l1, l1, eps));
    const R b2 = T::fma_(E2, E2, T::fma_(l2, l2, eps));
    R u0, u1, u2;
    if (sizeof(R) == 8) {
        const R t0 = b0 * b0, t1 = b1 * b1, t2 = b2 * b2;
        u0 = t1 * t2; u1 = t0 * t2; u2 = t0 * t1;
    } else {
        const float r0 = rcp_ulp((float)b0), r1 = rcp_ulp((float)b1), r2 = rcp_ulp((float)b2);
        u0 = r0 * r0; u1 = r1 * r1; u2 = r2 * r2;
    }
    const R a12 = T::fma_(R(2), u1, u2);
    den = T::fma_(R(1.0 / 3.0), u0, a12);
    num6s = T::fma_(a12, R(2) * Ta, -u2 * Tb);
    base6 = T::fma_(R(5 * WinScale<5>::iV), D1, R(-2 * WinScale<5>::iV) * D0);
}

// 2 F_hat at the interface whose newest needed cell sits in slot r of both windows (plus side lags one slot):
//   plus  side: cells i-3..i+3 = slots r-7..r-1, centre i   = V[r-4]
//   minus side: cells i-2..i+4 = slots r-6..r,   centre i+1 = V[r-3], stencil order reversed (D_j = -d[5-j], ...)
//   ORDER 5: plus cells i-2..i+2 = slots r-6..r-2 (centre V[r-4]); minus cells i-1..i+3 = slots r-5..r-1 reversed
// rot_flux_parts: 2 F_hat = vsum + corr / KW (KW = 12 for WENO7, 6 for WENO5) with vsum = 2 f+_i + 2 f-_{i+1} (twice the
// first-order Lax-Friedrichs flux) and corr / KW the high-order WENO correction (the limiter of R16 scales it by theta).
template <int r, int ORDER, typename R>
__device__ __forceinline__ void rot_flux_parts(const RotWin<R>& wp, const RotWin<R>& wm, R eps, R& vsum, R& corr) {
#define SL(k) (((r) + (k) + 16) & 7)
    R bp, np_, dp, bm, nm, dm;
    if (ORDER == 5) {
        weno5_diff<R>(wp.D[SL(-5)], wp.D[SL(-4)], wp.D[SL(-3)], wp.D[SL(-2)], wp.E[SL(-4)], wp.E[SL(-3)], wp.E[SL(-2)],
                      wp.G[SL(-3)], wp.G[SL(-2)], eps, bp, np_, dp);
        weno5_diff<R>(-wm.D[SL(-1)], -wm.D[SL(-2)], -wm.D[SL(-3)], -wm.D[SL(-4)], wm.E[SL(-1)], wm.E[SL(-2)], wm.E[SL(-3)],
                      -wm.G[SL(-1)], -wm.G[SL(-2)], eps, bm, nm, dm);
    } else {
    weno7_diff<R>(wp.D[SL(-6)], wp.D[SL(-5)], wp.D[SL(-4)],
                  wp.E[SL(-5)], wp.E[SL(-4)], wp.E[SL(-3)], wp.E[SL(-2)], wp.E[SL(-1)],
                  wp.S[SL(-4)], wp.S[SL(-3)], wp.S[SL(-2)], wp.S[SL(-1)],
                  wp.G[SL(-3)], wp.G[SL(-2)], wp.G[SL(-1)], bp, np_, dp);
    weno7_diff<R>(-wm.D[SL(0)], -wm.D[SL(-1)], -wm.D[SL(-2)],
                  wm.E[SL(0)], wm.E[SL(-1)], wm.E[SL(-2)], wm.E[SL(-3)], wm.E[SL(-4)],
                  wm.S[SL(0)], wm.S[SL(-1)], wm.S[SL(-2)], wm.S[SL(-3)],
                  wm.G[SL(0)], wm.G[SL(-1)], wm.G[SL(-2)], bm, nm, dm);
    }
    // xs = num+/den+ + num-/den- (WENO5: times sqrt(13)): one reciprocal for both sides in fp64
    R xs;
    if (sizeof(R) == 8) xs = (R)(fma((double)np_, (double)dm, (double)nm * (double)dp) * rcp_cubic((double)dp * (double)dm));
    else xs = (R)fmaf((float)np_, rcp_ulp((float)dp), (float)nm * rcp_ulp((float)dm));
    // KW x (high-order correction), KW = 12 or 6
    corr = ORDER == 5 ? Real<R>::fma_(R(WinScale<5>::iE), xs, bp + bm) : xs + (bp + bm);
    vsum = wp.V[SL(-4)] + wm.V[SL(-3)];                                       // WENO5: times sV
#undef SL
}
// KW x (2 F_hat) = KW vsum + corr, KW = 12 (WENO7) or 6 (WENO5): the 1/KW is folded into the divergence coefficient
template <int r, int ORDER, typename R>
__device__ __forceinline__ R rot_flux(const RotWin<R>& wp, const RotWin<R>& wm, R eps) {
    R vsum, corr;
    rot_flux_parts<r, ORDER, R>(wp, wm, eps, vsum, corr);
    return Real<R>::fma_(R(ORDER == 5 ? 6 * WinScale<5>::iV : 12), vsum, corr);
}

// per-thread view of one input stage: element pointers with the lane offset folded in
template <int DIR, typename R>
struct RowPtr {
    static constexpr int NCLS = DIR == 0 ? (sizeof(R) == 8 ? 4 : 2) : 1;      // DIR 0: one pointer per swizzle class
    const R* q[NCLS];
    __device__ __forceinline__ void set(const R* tile, int lane) {
        if (DIR == 0) {
#pragma unroll
            for (int k = 0; k < NCLS; ++k)
                q[k] = tile + lane * 8 + (sizeof(R) == 8 ? ((k ^ ((lane >> 1) & 3)) << 1) : ((k ^ ((lane >> 2) & 1)) << 2));
        } else q[0] = tile + lane;
    }
    template <int r>
    __device__ __forceinline__ R at() const {
        if (DIR == 0) return sizeof(R) == 8 ? q[(r >> 1) % NCLS][r & 1] : q[(r >> 2) % NCLS][r & 3];
        return q[0][r * 32];
    }
    // x sweeps, fp64: march cells r (even) and r + 1 of this lane as one 16-byte load (they share a chunk of the swizzled tile)
    template <int r>
    __device__ __forceinline__ double2 at2() const {
        static_assert(DIR == 0 && (r & 1) == 0, "row pairs exist in the x tiles only");
        return *reinterpret_cast<const double2*>(q[(r >> 1) % NCLS]);
    }
};

// ------------------------------------------------------------------------------------------------ limiter (R16, f-1)
// theta of one cell for the face state W1 = W0 + ks * c (W0 = U^L of the cell, c = the face's correction in the exchange
// tile, ks = +-6 dt/dx / (2 KW)): 1 if g(W1) >= delta, else (g(W0) - delta) / (g(W0) - g(W1)), g = E - |M|,
// delta = min(1e-8 E0, g(W0)).  Common case, decided on squares without looking at g(W0): delta <= 1e-8 E0, so
// g(W1) >= 1e-8 E0 already gives theta = 1.
template <typename R>
__device__ __forceinline__ R theta_cell(const R W0[4], const R c[4], R ks) {
    const R E0 = W0[0];
    const R d8 = R(1e-8) * E0;
    const R W1[4] = {Real<R>::fma_(ks, c[0], W0[0]), Real<R>::fma_(ks, c[1], W0[1]), Real<R>::fma_(ks, c[2], W0[2]),
                     Real<R>::fma_(ks, c[3], W0[3])};
    const R M12 = W1[1] * W1[1] + W1[2] * W1[2] + W1[3] * W1[3];
    const R t1 = W1[0] - d8;
    if (t1 >= R(0) && t1 * t1 >= M12) return R(1);
    const R M02 = W0[1] * W0[1] + W0[2] * W0[2] + W0[3] * W0[3];
    const R g0 = E0 - Real<R>::sqrt_(M02), g1 = W1[0] - Real<R>::sqrt_(M12);
    const R delta = d8 < g0 ? d8 : g0;
    if (g1 >= delta) return R(1);
    R t = (g0 - delta) / (g0 - g1);
    if (!(t >= R(0))) t = R(0);
    return t < R(1) ? t : R(1);
}

// theta of the face of chunk row r (between march cells i = cm + r - 4 and i + 1) for this lane: reads the corrections of
// the four energy-momentum fields from the chunk's output tiles (where phase A left them) and U^L of the two cells from
// the two U^L tiles (rows r-4, r-3; the previous chunk's tile for negative rows).  Cells outside the grid impose no
// condition.  Returns 1 if theta < 1.  r is a RUN-TIME argument on purpose: every warp calls this for its two rows, and
// eight compile-time copies (each with two divisions and two square roots on its slow path) made the limiter kernels
// instruction-cache bound (ncu r2_d: 40 % of the issue cycles stalled on "no instruction").
template <int DIR, int NF, typename R>
__device__ __noinline__ int theta_row(int r, const R* st, const R* stp, const R* xc_all, R* th, int lane, int cm, int nd, R k3lam) {
    const int o = sub_off<DIR, R>(r, lane);
    R a[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) a[q] = xc_all[q * RING_SUB + o];
    const int i = cm + r - 4;
    R theta = R(1);
    if (i >= 0 && i <= nd - 1) {
        const int rl = (r + 4) & 7;
        const R* s = r < 4 ? stp : st;
        const int ol = sub_off<DIR, R>(rl, lane);
        const R W0[4] = {s[ol], s[RING_SUB + ol], s[2 * RING_SUB + ol], s[3 * RING_SUB + ol]};
        const R t = theta_cell<R>(W0, a, -k3lam);
        theta = t < theta ? t : theta;
    }
    if (i + 1 >= 0 && i + 1 <= nd - 1) {
        const int rr = (r + 5) & 7;
        const R* s = r < 3 ? stp : st;
        const int orr = sub_off<DIR, R>(rr, lane);
        const R W0[4] = {s[orr], s[RING_SUB + orr], s[2 * RING_SUB + orr], s[3 * RING_SUB + orr]};
        const R t = theta_cell<R>(W0, a, k3lam);
        theta = t < theta ? t : theta;
    }
    th[o] = theta;
    return theta < R(1) ? 1 : 0;
}

// x sweeps: theta of the faces of chunk rows r0 (even) and r0 + 1 together.  In the swizzled x tiles a lane's march cells
// r0, r0 + 1 share one 16-byte chunk, and a warp's 8-byte loads of ONE row are 2-way bank conflicted whatever the swizzle
// (all lanes read the same half of their 16-byte chunk: ncu counts 48-53e6 conflicts in 102-111e6 shared-memory wavefronts
// of the limiter x kernels and 0.9-1.0 short-scoreboard stall cycles per issued instruction, against 0.44 in y/z), while
// 16-byte loads of a row PAIR are conflict-free: 12 loads (8 of them pairs) instead of 24 for the two faces.
template <int NF>
__device__ __noinline__ int theta_rows2_x(int r0, const double* st, const double* stp, const double* xc_all, double* th, int lane,
                                          int cm, int nd, double k3lam) {
    const int sw = (lane >> 1) & 3;
    const int o2 = lane * 8 + (((r0 >> 1) ^ sw) << 1);                     // rows r0, r0 + 1 of this lane
    double2 c[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) c[q] = *reinterpret_cast<const double2*>(xc_all + q * RING_SUB + o2);
    // U^L of the cells i0 = cm + r0 - 4, i0 + 1 (rows (r0 + 4) & 7, + 1: one pair) and i0 + 2 (row (r0 + 6) & 7)
    const int i0 = cm + r0 - 4;
    const double* sa = r0 < 4 ? stp : st;
    const int oa = lane * 8 + (((((r0 + 4) & 7) >> 1) ^ sw) << 1);
    const double* sc = r0 < 2 ? stp : st;
    const int oc = lane * 8 + (((((r0 + 6) & 7) >> 1) ^ sw) << 1);
    double2 ua[4];
    double uc[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        ua[q] = *reinterpret_cast<const double2*>(sa + q * RING_SUB + oa);
        uc[q] = sc[q * RING_SUB + oc];
    }
    const double A[4] = {ua[0].x, ua[1].x, ua[2].x, ua[3].x}, B[4] = {ua[0].y, ua[1].y, ua[2].y, ua[3].y};
    const double c0[4] = {c[0].x, c[1].x, c[2].x, c[3].x}, c1[4] = {c[0].y, c[1].y, c[2].y, c[3].y};
    double t0 = 1.0, t1 = 1.0;
    if (i0 >= 0 && i0 <= nd - 1) { const double t = theta_cell<double>(A, c0, -k3lam); t0 = t < t0 ? t : t0; }
    if (i0 + 1 >= 0 && i0 + 1 <= nd - 1) {
        double t = theta_cell<double>(B, c0, k3lam);
        t0 = t < t0 ? t : t0;
        t = theta_cell<double>(B, c1, -k3lam);
        t1 = t < t1 ? t : t1;
    }
    if (i0 + 2 >= 0 && i0 + 2 <= nd - 1) { const double t = theta_cell<double>(uc, c1, k3lam); t1 = t < t1 ? t : t1; }
    *reinterpret_cast<double2*>(th + o2) = make_double2(t0, t1);
    return (t0 < 1.0 ? 1 : 0) + (t1 < 1.0 ? 1 : 0);
}

template <typename R, int ORDER, int LIM, int DIR, int OUT, int NF>
struct SweepCtx {
    RotWin<R> wp, wm;
    R fhat_prev;
    R corr_even;                           // limiter x sweeps, phase A: the even row's correction waits for the odd row's
    const R* th;                           // limiter: theta tile
    R alpha, eps, coef, rk_a, rk_b;           // coef: everything that multiplies (F_hat_prev - F_hat), see the kernel
    // current chunk
    RowPtr<DIR, R> pu, pmd, pw, pp;        // own field, normal momentum, W (energy: zeros), P (energy: M_d; else zeros)
    RowPtr<DIR, R> pus[2];                 // U_s of the output cells: rows 4..7 of the previous chunk, 0..3 of this one
    RowPtr<DIR, R> pun;                    // U^n of the output cells
    R* out;                                // this field's output sub-tile, lane offset NOT folded in
    int lane;

    // split fluxes of the row's cell, carried as 2 f^+- = F +- alpha U:
    //   F^d_E = M_d;  F^d_{M_j} = M_j v_d + p delta_jd;  F^d_{N_B} = N_B v_d;  v_d = M_d * W   (a-3)
    // written branch-free as F = U_f * (M_d * W') + C with per-warp operand tiles: momenta / N_B: W' = W, C = p (normal
    // component) or a tile of zeros; energy: W' = zeros, C = M_d (E * 0 + M_d: four shared-memory loads per row, not five).
    struct RowIn { R u, md, w, p; };
    template <int r>
    __device__ __forceinline__ void load(RowIn& in) const {
        in.u = pu.template at<r>();
        in.md = pmd.template at<r>();
        in.w = pw.template at<r>();
        in.p = pp.template at<r>();
    }
    template <int r>
    __device__ __forceinline__ void push(const RowIn& in) {
        typedef Real<R> T;
        const R B = in.md * in.w;
        R F = T::fma_(in.u, B, in.p);
        if (ORDER == 5) F *= R(WinScale<5>::sV);             // alpha carries the same factor
        rot_push<r, ORDER, R>(wp, T::fma_(alpha, in.u, F), eps);
        rot_push<r, ORDER, R>(wm, T::fma_(-alpha, in.u, F), eps);
    }
    template <int r>
    __device__ __forceinline__ void load_push() {
        RowIn in;
        load<r>(in);
        push<r>(in);
    }
    // The 8 rows of a chunk, software-pipelined by hand: the shared-memory loads of row r+1 are issued BEFORE row r
    // is emitted -- the compiler cannot move a load above the output-tile store (it cannot prove they do not alias), so
    // in source order "load, compute, store" per row every row would start with an exposed load latency and end with
    // the serial reciprocal chain.  MODE 0: emit<r>(); MODE 1: limiter phase A (corr_store).
    template <int MODE, int r>
    __device__ __forceinline__ void tail(const RowIn& in) {
        push<r>(in);
        if (MODE == 0) emit<r>();
        else corr_tail<r>();
    }
    template <int MODE>
    __device__ __forceinline__ void rows() {
        RowIn i0, i1;
        if (sizeof(R) == 8 && NF == 5) {
            // nf = 5 in fp64 is compiled for <= 136 registers (3 blocks of 160 threads): the extra live row does not fit
            load<0>(i0); tail<MODE, 0>(i0); load<1>(i0); tail<MODE, 1>(i0); load<2>(i0); tail<MODE, 2>(i0);
            load<3>(i0); tail<MODE, 3>(i0); load<4>(i0); tail<MODE, 4>(i0); load<5>(i0); tail<MODE, 5>(i0);
            load<6>(i0); tail<MODE, 6>(i0); load<7>(i0); tail<MODE, 7>(i0);
            return;
        }
        load<0>(i0);
        load<1>(i1); tail<MODE, 0>(i0);
        load<2>(i0); tail<MODE, 1>(i1);
        load<3>(i1); tail<MODE, 2>(i0);
        load<4>(i0); tail<MODE, 3>(i1);
        load<5>(i1); tail<MODE, 4>(i0);
        load<6>(i0); tail<MODE, 5>(i1);
        load<7>(i1); tail<MODE, 6>(i0);
        tail<MODE, 7>(i1);
    }
    // limiter, phase A: the row's high-order correction goes to the exchange tile
    template <int r>
    __device__ __forceinline__ void corr_tail() {
        R vsum, corr;
        rot_flux_parts<r, ORDER, R>(wp, wm, eps, vsum, corr);
        if constexpr (DIR == 0 && sizeof(R) == 8 && RING_LIM_X_PAIRS > 2) {
            // x tiles: rows r - 1, r as one 16-byte store (an 8-byte store of one row is 2-way bank conflicted)
            if (r & 1) *reinterpret_cast<double2*>(out + sub_off<DIR, R>(r - 1, lane)) = make_double2((double)corr_even, (double)corr);
            else corr_even = corr;
        } else
        out[sub_off<DIR, R>(r, lane)] = corr;                // phase A leaves the correction where the output will go
    }
    // limiter, phase C: the first-order part of every flux is already inside U^L; what is left is theta * corr
    template <int r>
    __device__ __forceinline__ void emit_lim() {
        const int o = sub_off<DIR, R>(r, lane);
        emit_with<r>(th[o] * out[o]);
    }
    // the same for rows r (even) and r + 1 of an x sweep from 16-byte loads and one 16-byte store (conflict-free, see
    // theta_rows2_x); the arithmetic is emit_with's, operation by operation
    template <int r>
    __device__ __forceinline__ void emit_lim2() {
        if constexpr (DIR == 0 && sizeof(R) == 8) {
            const int o = sub_off<DIR, R>(r, lane);
            const double2 t = *reinterpret_cast<const double2*>(th + o);
            const double2 c = *reinterpret_cast<const double2*>(out + o);
            const double f0 = t.x * c.x, f1 = t.y * c.y;
            const double d0 = fhat_prev - f0, d1 = f0 - f1;
            fhat_prev = f1;
            double2 w;
            if (OUT == OUT_STORE || OUT == OUT_REDUCE) { w.x = d0 * coef; w.y = d1 * coef; }
            else {
                const double2 us = pus[r < 4 ? 0 : 1].template at2<(r + 4) & 7>();
                if (OUT == OUT_COMBINE) {
                    const double2 un = pun.template at2<r>();
                    w.x = fma(coef, d0, fma(rk_b, us.x, rk_a * un.x));
                    w.y = fma(coef, d1, fma(rk_b, us.y, rk_a * un.y));
                } else { w.x = fma(coef, d0, us.x); w.y = fma(coef, d1, us.y); }
            }
            *reinterpret_cast<double2*>(out + o) = w;
        }
    }
    template <int r>
    __device__ __forceinline__ void emit() {
        emit_with<r>(rot_flux<r, ORDER, R>(wp, wm, eps));
    }
    template <int r>
    __device__ __forceinline__ void emit_with(const R fhat) {
        typedef Real<R> T;
        const R dlt = fhat_prev - fhat;
        fhat_prev = fhat;
        R o;
        if (OUT == OUT_STORE || OUT == OUT_REDUCE) o = dlt * coef;
        else {
            // output cell i = (row's cell) - 4: U_s from the ring, row (r + 4) & 7 of the previous / this chunk
            const R us = pus[r < 4 ? 0 : 1].template at<(r + 4) & 7>();
            if (OUT == OUT_COMBINE) o = T::fma_(coef, dlt, T::fma_(rk_b, us, rk_a * pun.template at<r>()));
            else o = T::fma_(coef, dlt, us);
        }
        out[sub_off<DIR, R>(r, lane)] = o;
    }
};

template <typename R, int ORDER, int LIM, int DIR, int OUT, int NF>
__global__ void __launch_bounds__(32 * NF, ring_blocks_per_sm(NF, sizeof(R), OUT, LIM))
k_sweep_ring(const __grid_constant__ RingMaps maps, const RingArgs a) {
    // 1024-byte alignment: the swizzle pattern is a function of the absolute shared address
    extern __shared__ __align__(1024) unsigned char smem[];
    constexpr int STAGE_REALS = ring_stage_reals(NF, LIM);
    constexpr uint32_t STAGE_BYTES = STAGE_REALS * sizeof(R);
    constexpr uint32_t UN_BYTES = NF * RING_SUB * sizeof(R);
    R* stages = (R*)smem;
    constexpr int NSTAGE = ring_nstage(OUT, LIM);
    R* outt = stages + NSTAGE * STAGE_REALS;                           // two output tiles of NF sub-tiles
    R* unt = outt + 2 * NF * RING_SUB;                                 // OUT_COMBINE: two U^n tiles (limiter: one)
    R* zeros = unt + (OUT == OUT_COMBINE ? (LIM ? 1 : 2) * NF * RING_SUB : 0);
    R* ult = zeros + RING_SUB;                                         // limiter: two U^L tiles of NF sub-tiles, then the theta tile
    R* tht = ult + (LIM ? 2 * NF * RING_SUB : 0);
    uint64_t* full = (uint64_t*)(tht + (LIM ? RING_SUB : 0));
    uint64_t* full_ul = full + RING_NSTAGE_MAX;
    uint64_t* full_un = full_ul + 2;                                   // limiter + OUT_COMBINE: the single U^n tile

    // NF = 1: the baryon density N_B (field 4) of a 5-field state on its own, F = N_B v_d: a one-warp block whose stage
    // holds [N_B][W][M_d] (M_d in the slot P has otherwise).  With the 4-warp kernel on fields 0..3 it replaces the 5-warp
    // kernel in fp64, whose 160-thread blocks cannot hold the pipelined row loop at 3 blocks/SM.
    constexpr bool BARYON = (NF == 1);
    constexpr int F0 = BARYON ? 4 : 0;                                 // first field of the boxes
    static_assert(!(BARYON && LIM), "the limiter needs all energy-momentum fields in one block");
    const int lane = threadIdx.x, f = threadIdx.y;
    const bool leader = (lane == 0 && f == 0);
    const int nd = DIR == 0 ? a.nx : DIR == 1 ? a.ny : a.nz;

    // transverse tile of 32 lines and the march segment of this block.  Uniform mode (n_long < 0): blockIdx.x = tile,
    // blockIdx.y = segment of seg_len cells.  Tail-split mode: the first n_long tiles are marched whole by one block each
    // (they fill complete waves of resident blocks); the remaining tiles are cut into short_nseg segments of short_len
    // cells so that the last, partial wave is made of short blocks.
    int tile, s0, seglen;
    if (a.n_long < 0) { tile = blockIdx.x; s0 = blockIdx.y * a.seg_len; seglen = a.seg_len; }
    else if ((int)blockIdx.x < a.n_long) { tile = blockIdx.x; s0 = 0; seglen = nd; }
    else {
        const int bb = blockIdx.x - a.n_long;
        tile = a.n_long + bb / a.short_nseg;
        s0 = (bb % a.short_nseg) * a.short_len;
        seglen = a.short_len;
    }
    int t0, tfix;                  // first transverse index along the lane axis, fixed transverse index
    {
        const int nlane_axis = DIR == 0 ? a.ny : a.nx;
        const int tiles = (nlane_axis + 31) >> 5;
        const int tb = tile % tiles;
        tfix = tile / tiles;
        t0 = tb << 5;
    }
    if (s0 >= nd) return;          // whole block exits together
    const int len = min(nd, s0 + seglen) - s0;
    const int nchunks = (len + RING_CH - 1) / RING_CH + 1;             // chunk m holds cells s0 - 4 + 8m .. + 7

    if (leader) {
#pragma unroll
        for (int s = 0; s < NSTAGE; ++s) mbar_init(&full[s], 1);
        if (LIM) { mbar_init(&full_ul[0], 1); mbar_init(&full_ul[1], 1); mbar_init(full_un, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = f * 32 + lane; i < RING_SUB; i += 32 * NF) zeros[i] = R(0);
    __syncthreads();

    auto coords = [&](int cm, int& c0, int& c1, int& c2) {
        if (DIR == 0) { c0 = cm; c1 = t0; c2 = tfix; }
        else if (DIR == 1) { c0 = t0; c1 = cm; c2 = tfix; }
        else { c0 = t0; c1 = tfix; c2 = cm; }
    };
    auto issue = [&](int m) {                                          // leader only
        const int st = m % NSTAGE;
        R* dst = stages + st * STAGE_REALS;
        int c0, c1, c2;
        coords(s0 - 4 + m * RING_CH, c0, c1, c2);
        const bool with_un = (OUT == OUT_COMBINE) && !LIM && m > 0;
        mbar_expect_tx(&full[st], STAGE_BYTES + (with_un ? UN_BYTES : 0u));
        tma_load_4d(dst, &maps.U, &full[st], c0, c1, c2, F0);
        tma_load_4d(dst + NF * RING_SUB, &maps.W, &full[st], c0, c1, c2, 0);
        if (BARYON) tma_load_4d(dst + (NF + 1) * RING_SUB, &maps.U, &full[st], c0, c1, c2, 1 + DIR);
        else tma_load_4d(dst + (NF + 1) * RING_SUB, &maps.P, &full[st], c0, c1, c2, 0);
        if (with_un) {
            coords(s0 + (m - 1) * RING_CH, c0, c1, c2);                // the cells chunk m emits
            tma_load_4d(unt + (m & 1) * NF * RING_SUB, &maps.Un, &full[st], c0, c1, c2, F0);
        }
    };
    auto issue_ul = [&](int m) {                                       // leader only (limiter): U^L of chunk m's cells
        int c0, c1, c2;
        coords(s0 - 4 + m * RING_CH, c0, c1, c2);
        mbar_expect_tx(&full_ul[m & 1], UN_BYTES);
        tma_load_4d(ult + (m & 1) * NF * RING_SUB, &maps.UL, &full_ul[m & 1], c0, c1, c2, 0);
    };
    // limiter + OUT_COMBINE: U^n of the cells chunk m emits into the one U^n tile, issued at the top of chunk m (phase C of
    // chunk m-1 was its last reader) and needed only in phase C, a whole phase A later
    auto issue_un = [&](int m) {                                       // leader only
        int c0, c1, c2;
        coords(s0 + (m - 1) * RING_CH, c0, c1, c2);
        mbar_expect_tx(full_un, UN_BYTES);
        tma_load_4d(unt, &maps.Un, full_un, c0, c1, c2, F0);
    };
    auto flush = [&](int m) {                                          // leader only: write back chunk m's outputs
        int c0, c1, c2;
        coords(s0 + (m - 1) * RING_CH, c0, c1, c2);
        const R* src = outt + (m & 1) * NF * RING_SUB;
        if (OUT == OUT_REDUCE) tma_reduce_add_4d(&maps.Out, src, c0, c1, c2, F0);
        else tma_store_4d(&maps.Out, src, c0, c1, c2, F0);
        tma_commit();
    };
    if (leader) {
        issue(0);
        if (nchunks > 1) issue(1);
        if (LIM) issue_ul(0);
    }

    SweepCtx<R, ORDER, LIM, DIR, OUT, NF> cx;
    cx.th = tht;
    int nlim_local = 0;
    cx.wp.clear();
    cx.wm.clear();
    cx.fhat_prev = R(0);
    cx.alpha = Real<R>::from_bits(a.diag->slot[a.slot].alpha_bits[DIR]) * R(WinScale<ORDER>::sV);
    cx.eps = (R)a.eps_eff;
    {
        // the fluxes are carried as KW x 2 F_hat (KW = 12, 6: rot_flux); c = a.coef / KW turns their difference into the
        // divergence part; the COMBINE kernels fold dt (and the RK weight b) in: U_next = a U^n + b U_s + (b dt c) (F- - F+)
        const double c = a.coef / (ORDER == 5 ? 6.0 : 12.0);
        cx.coef = (R)(OUT == OUT_COMBINE ? a.rk_b * a.dt * c : OUT == OUT_COMBINE1 ? a.dt * c : c);
    }
    cx.rk_a = (R)a.rk_a;
    cx.rk_b = (R)a.rk_b;
    cx.lane = lane;
    const bool is_energy = !BARYON && f == 0, is_normal = !BARYON && f == 1 + DIR;

    for (int m = 0; m < nchunks; ++m) {
        const int cm = s0 - 4 + m * RING_CH;
        if (m > 0) {
            fence_proxy_async();                                       // output-tile / fix-up writes -> async proxy
            if (leader) tma_wait_read0();                              // the write-back issued one chunk ago has read its tile
            __syncthreads();                                           // everyone is done with chunk m-1
            if (leader) {
                if (m > 1) flush(m - 1);
                if (m + 1 < nchunks) issue(m + 1);                     // overwrites chunk m+1-NSTAGE
                if (LIM) issue_ul(m);                                  // overwrites chunk m-2's U^L (phase B of m-1 is over)
                if (LIM && OUT == OUT_COMBINE) issue_un(m);
            }
        }
        R* st = stages + (m % NSTAGE) * STAGE_REALS;
        // chunk m-1; with two stages it is chunk m+1's target, but the only reader outside the 3-stage combine kernels is
        // the ghost fix-up of a line's LAST chunk, after which nothing is loaded
        const R* stp = stages + ((m + NSTAGE - 1) % NSTAGE) * STAGE_REALS;
        mbar_wait(&full[m % NSTAGE], (m / NSTAGE) & 1);

        // a-7: ghost rows (block-uniform test; at most the first and the last two chunks of a grid line)
        if (cm < 0 || cm + RING_CH - 1 > nd - 1) {
            const int rlast = nd - 1 - cm;                             // row of the last interior cell (may be < 0)
            for (int t = f; t < NF + 2; t += NF) {
#pragma unroll
                for (int r = 0; r < RING_CH; ++r) {
                    const int c = cm + r;
                    if (c < 0) st[t * RING_SUB + sub_off<DIR, R>(r, lane)] = st[t * RING_SUB + sub_off<DIR, R>(-cm, lane)];
                    else if (c > nd - 1) {
                        st[t * RING_SUB + sub_off<DIR, R>(r, lane)] =
                            rlast >= 0 ? st[t * RING_SUB + sub_off<DIR, R>(rlast, lane)]
                                       : stp[t * RING_SUB + sub_off<DIR, R>(rlast + RING_CH, lane)];
                    }
                }
            }
            __syncthreads();
        }

        cx.pu.set(st + f * RING_SUB, lane);
        cx.pmd.set(st + (BARYON ? NF + 1 : 1 + DIR) * RING_SUB, lane);
        cx.pw.set(is_energy ? zeros : st + NF * RING_SUB, lane);
        cx.pp.set(is_energy ? st + (1 + DIR) * RING_SUB : is_normal ? st + (NF + 1) * RING_SUB : zeros, lane);
        if (OUT == OUT_COMBINE1 || OUT == OUT_COMBINE) {           // the state the stage's own part is added to: U_s, or U^L
            cx.pus[0].set(LIM ? ult + ((m + 1) & 1) * NF * RING_SUB + f * RING_SUB : stp + f * RING_SUB, lane);
            cx.pus[1].set(LIM ? ult + (m & 1) * NF * RING_SUB + f * RING_SUB : st + f * RING_SUB, lane);
        }
        if (OUT == OUT_COMBINE) cx.pun.set(unt + (LIM ? 0 : (m & 1)) * NF * RING_SUB + f * RING_SUB, lane);
        cx.out = outt + (m & 1) * NF * RING_SUB + f * RING_SUB;

        const R* ul_cur = ult + (m & 1) * NF * RING_SUB;            // limiter: U^L tiles of this / the previous chunk
        const R* ul_prev = ult + ((m + 1) & 1) * NF * RING_SUB;
        const R* xcm = outt + (m & 1) * NF * RING_SUB;              // limiter: the corrections sit in the output tiles
        if (m == 0) {
            // warm-up chunk: cells s0-4 .. s0+3 fill both windows; the last row gives the interface s0 - 1/2
            cx.template load_push<0>(); cx.template load_push<1>(); cx.template load_push<2>(); cx.template load_push<3>();
            cx.template load_push<4>(); cx.template load_push<5>(); cx.template load_push<6>(); cx.template load_push<7>();
            if (!LIM) cx.fhat_prev = rot_flux<7, ORDER, R>(cx.wp, cx.wm, cx.eps);
            else {
                R vsum, corr;
                rot_flux_parts<7, ORDER, R>(cx.wp, cx.wm, cx.eps, vsum, corr);
                cx.out[sub_off<DIR, R>(7, lane)] = corr;
                mbar_wait(&full_ul[m & 1], (m >> 1) & 1);
                __syncthreads();
                if (f == 0) {
                    const int n1 = theta_row<DIR, NF, R>(7, ul_cur, ul_prev, xcm, tht, lane, cm, nd, (R)a.k3lam);
                    // inner segment starts are counted by the segment before; z sweep: the face below plane 0
                    if (s0 == 0 && (DIR == 2 ? a.own_lo == 0 : (tfix >= a.own_lo && tfix < a.own_hi))) nlim_local += n1;
                }
                __syncthreads();
                cx.fhat_prev = tht[sub_off<DIR, R>(7, lane)] * corr;
            }
        } else if (!LIM) {
            cx.template rows<0>();
        } else {
            // R16: (A) corrections of all fields to shared memory, (B) one theta per face from all fields, (C) emit
            cx.template rows<1>();
            mbar_wait(&full_ul[m & 1], (m >> 1) & 1);
            __syncthreads();
            const R k3 = (R)a.k3lam;
            int n0 = 0, n1 = 0;
            if (f < 4) {                                            // warp f: the faces of rows 2f and 2f + 1
                if constexpr (DIR == 0 && sizeof(R) == 8 && RING_LIM_X_PAIRS) {
                    n0 = theta_rows2_x<NF>(2 * f, (const double*)ul_cur, (const double*)ul_prev, (const double*)xcm, (double*)tht,
                                           lane, cm, nd, (double)k3);   // both faces; x sweep: one ownership test serves both
                } else {
                    n0 = theta_row<DIR, NF, R>(2 * f, ul_cur, ul_prev, xcm, tht, lane, cm, nd, k3);
                    n1 = theta_row<DIR, NF, R>(2 * f + 1, ul_cur, ul_prev, xcm, tht, lane, cm, nd, k3);
                }
            }
            if (n0 | n1) {                                          // rare: only now look at ownership (z-slabs)
                const int il = cm + 2 * f - 4;                      // faces of rows 2f, 2f+1: lower cells il, il + 1
                const bool cnt0 = DIR == 2 ? (il >= a.own_lo && il < a.own_hi) : (tfix >= a.own_lo && tfix < a.own_hi);
                const bool cnt1 = DIR == 2 ? (il + 1 >= a.own_lo && il + 1 < a.own_hi) : cnt0;
                nlim_local += (cnt0 ? n0 : 0) + (cnt1 ? n1 : 0);
            }
            if (OUT == OUT_COMBINE) mbar_wait(full_un, (m - 1) & 1);
            __syncthreads();
            if constexpr (DIR == 0 && sizeof(R) == 8 && RING_LIM_X_PAIRS > 1) {
                cx.template emit_lim2<0>(); cx.template emit_lim2<2>(); cx.template emit_lim2<4>(); cx.template emit_lim2<6>();
            } else {
                cx.template emit_lim<0>(); cx.template emit_lim<1>(); cx.template emit_lim<2>(); cx.template emit_lim<3>();
                cx.template emit_lim<4>(); cx.template emit_lim<5>(); cx.template emit_lim<6>(); cx.template emit_lim<7>();
            }
        }
    }
    fence_proxy_async();
    if (leader) tma_wait_read0();
    __syncthreads();
    if (leader) {
        if (nchunks > 1) flush(nchunks - 1);
        tma_wait_all0();
    }
    if (LIM) {
        for (int off = 16; off > 0; off >>= 1) nlim_local += __shfl_xor_sync(0xffffffffu, nlim_local, off);
        if (lane == 0 && nlim_local) atomicAdd(a.nlim, (unsigned long long)nlim_local);
    }
}

}  // namespace hydro_dev
