// hydro_sweep_tma.cuh -- the WENO7-LF sweep kernels of the hot path, TMA-staged (sm_100a).  PRODUCT.
//
// Same arithmetic as k_sweep (hydro_kernels.cuh: a-3 WENO7 reconstruction of the Lax-Friedrichs split fluxes,
// a-4 flux divergence, a-6 stage combination, a-7 outflow ghosts), different data movement:
//
//   block  = 32 lanes x NF field-warps.  The 32 lanes are 32 neighbouring grid lines (consecutive x for the y/z
//            sweeps, consecutive y for the x sweep); warp f reconstructs conserved field f, so the four (five)
//            warps of a block share every input row: U (all fields), W = scale/(E+p) and P.
//   input  = a ring of NSTAGE shared-memory stages, each holding CH = 8 march cells x 32 lanes of (U[NF], W, P),
//            filled by ONE thread with three cp.async.bulk.tensor (TMA) box loads per stage that complete on an
//            mbarrier; loads run NSTAGE-1 chunks (24 march cells) ahead of the arithmetic, which removes the
//            long-scoreboard stalls of the direct-load kernel (profiles/r1_a_*: FP64 pipe 34 % busy).
//   x sweep: the box is (8 cells along x) x (32 rows of y) with the 64-byte TMA swizzle, so that lane = row reads
//            its own row from shared memory (2-way bank conflict) instead of 32 scattered global sectors, and the
//            -div tile goes back through a swizzled shared tile and a TMA box store (coalesced along x).
//   ghosts : TMA zero-fills out-of-range cells; the outflow clamp is applied when the row is consumed (low end:
//            read the row of cell 0, which sits in the first chunk; high end: keep the last valid split fluxes).
#pragma once
#include <cuda.h>
#include "hydro_kernels.cuh"

namespace hydro_dev {

constexpr int TMA_CH = 8;          // march cells per chunk
constexpr int TMA_NSTAGE = 4;      // ring depth
constexpr int TMA_SUB = TMA_CH * 32;   // reals per sub-tile (one field, one chunk)

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
    for (unsigned spin = 0; spin < (1u << 20); ++spin) {
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
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// shared-memory bytes of one launch (host and device agree through this function)
__host__ __device__ constexpr int sweep_tma_stage_reals(int nf) { return (nf + 2) * TMA_SUB; }
__host__ __device__ constexpr int sweep_tma_smem_bytes(int nf, int dir, int esz) {
    return TMA_NSTAGE * sweep_tma_stage_reals(nf) * esz + (dir == 0 ? 2 * nf * TMA_SUB * esz : 0) + 64 + 1024;
}

struct SweepMaps {
    CUtensorMap U, W, P, Lst;      // loads of the stage state, W, P; store of the -div tile (x sweep only)
};

// element offset inside a sub-tile of march row r (0..7) for this lane
template <int DIR>
__device__ __forceinline__ int sub_off(int r, int lane) {
    if (DIR == 0) {
        // dense box layout (8 cells of x fastest, 32 rows): byte = lane*64 + r*8, TMA 64-byte swizzle:
        // 16-byte chunk index (bits 4..5) ^= address bits 7..8 = (lane >> 1) & 3
        return lane * 8 + ((((r >> 1) ^ ((lane >> 1) & 3)) << 1) | (r & 1));
    }
    return r * 32 + lane;
}

// MODE as in k_sweep: 0: L = -D_d;  1: L -= D_d;  2: U_next = a U^n + b (U_s + dt (L - D_d))
template <int DIR, int MODE, int NF>
__global__ void __launch_bounds__(32 * NF, NF == 4 ? 3 : 2)
k_sweep_tma(const __grid_constant__ SweepMaps maps, SweepArgs<double> a) {
    typedef double R;
    typedef Real<R> T;
    extern __shared__ unsigned char smem_raw[];
    // 1024-byte alignment: the swizzle pattern is a function of the absolute shared address
    unsigned char* smem = (unsigned char*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    constexpr int STAGE_REALS = sweep_tma_stage_reals(NF);
    constexpr uint32_t STAGE_BYTES = STAGE_REALS * sizeof(R);
    R* stages = (R*)smem;
    R* outt = stages + TMA_NSTAGE * STAGE_REALS;                       // DIR 0: two -div tiles of NF sub-tiles
    uint64_t* full = (uint64_t*)(outt + (DIR == 0 ? 2 * NF * TMA_SUB : 0));

    const int lane = threadIdx.x, f = threadIdx.y;
    const bool leader = (lane == 0 && f == 0);
    const int nd = DIR == 0 ? a.nx : DIR == 1 ? a.ny : a.nz;

    // transverse tile of 32 lines and the march segment of this block
    int t0, tfix;                  // first transverse index along the lane axis, fixed transverse index
    {
        const int nlane_axis = DIR == 0 ? a.ny : a.nx;
        const int tiles = (nlane_axis + 31) >> 5;
        const int tb = blockIdx.x % tiles;
        tfix = blockIdx.x / tiles;
        t0 = tb << 5;
    }
    const int ls = a.seg_len;
    const int s0 = blockIdx.y * ls;
    const int s1 = min(nd, s0 + ls);
    if (s0 >= s1) return;          // whole block exits together
    const int len = s1 - s0;
    const int nchunks = (len + 8 + TMA_CH - 1) / TMA_CH;
    const bool valid = (t0 + lane) < (DIR == 0 ? a.ny : a.nx);

    if (leader) {
#pragma unroll
        for (int s = 0; s < TMA_NSTAGE; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto issue = [&](int m) {
        const int st = m % TMA_NSTAGE;
        R* dst = stages + st * STAGE_REALS;
        const int cm = s0 - 4 + m * TMA_CH;
        int c0, c1, c2;
        if (DIR == 0) { c0 = cm; c1 = t0; c2 = tfix; }
        else if (DIR == 1) { c0 = t0; c1 = cm; c2 = tfix; }
        else { c0 = t0; c1 = tfix; c2 = cm; }
        mbar_expect_tx(&full[st], STAGE_BYTES);
        tma_load_4d(dst, &maps.U, &full[st], c0, c1, c2, 0);
        tma_load_4d(dst + NF * TMA_SUB, &maps.W, &full[st], c0, c1, c2, 0);
        tma_load_4d(dst + (NF + 1) * TMA_SUB, &maps.P, &full[st], c0, c1, c2, 0);
    };
    if (leader) {
        for (int m = 0; m < TMA_NSTAGE && m < nchunks; ++m) issue(m);      // the ring starts full
    }

    const R alpha = T::from_bits(a.diag->slot[a.slot].alpha_bits[DIR]);
    const R c3 = R(39.05), eps = a.eps_eff;
    const bool is_energy = (f == 0), is_normal = (f == 1 + DIR);

    // global addressing of this thread's line (y/z sweeps store directly; coalesced over the 32 lanes)
    long long base = 0, stride = 0;
    if (DIR == 1) { base = (long long)tfix * a.nx * a.ny + (t0 + lane); stride = a.nx; }
    if (DIR == 2) { base = (long long)tfix * a.nx + (t0 + lane); stride = (long long)a.nx * a.ny; }
    R* __restrict__ Lf = a.L + (long long)f * a.N;
    const R* __restrict__ Unf = a.use_un ? a.Un + (long long)f * a.N : a.U;
    R* __restrict__ Uof = a.Uout + (long long)f * a.N;

    Win<R> wp, wm;
    wp.clear();
    wm.clear();
    R fp_pending = R(0), fp2 = R(0), fm2 = R(0), ucell[TMA_CH];
    R fhat_prev = R(0);
    R lpre = R(0), upre = R(0);                                      // L / U^n of the next cell to emit (prefetch)

    // split flux of march cell c from stage row `row` (carried as 2 f^+- = F +- alpha U)
    auto load_row = [&](const R* st, int row, R& u_out) {
        const int o = sub_off<DIR>(row, lane);
        const R u = st[f * TMA_SUB + o];
        const R md = st[(1 + DIR) * TMA_SUB + o];
        R F;
        if (is_energy) F = md;                                       // F^d_E = M_d
        else {
            const R vd = md * st[NF * TMA_SUB + o];
            F = u * vd;                                              // M_j v_d, N_B v_d
            if (is_normal) F += st[(NF + 1) * TMA_SUB + o];          // + p delta_jd
        }
        fp2 = T::fma_(alpha, u, F);
        fm2 = T::fma_(-alpha, u, F);
        u_out = u;
    };

    int q = 0;                                                       // stream position: march cell c = s0 - 4 + q
    for (int m = 0; m < nchunks; ++m) {
        if (m > 0) {
            if (DIR == 0) {
                fence_proxy_async();                                 // -div tile writes -> visible to the TMA store
                if (leader) tma_wait_read0();                        // the store issued one chunk ago has read its tile
            }
            __syncthreads();                                         // everyone is done with chunk m-1
            if (leader) {
                if (DIR == 0 && m > 1) {                             // chunk m-1 emitted cells s0 + (m-2)*8 ..
                    const R* src = outt + ((m - 1) & 1) * NF * TMA_SUB;
                    tma_store_4d(&maps.Lst, src, s0 + (m - 2) * TMA_CH, t0, tfix, 0);
                    tma_commit();
                }
                if (m + TMA_NSTAGE - 1 < nchunks) issue(m + TMA_NSTAGE - 1);
            }
        }
        const R* st = stages + (m % TMA_NSTAGE) * STAGE_REALS;
        mbar_wait(&full[m % TMA_NSTAGE], (m / TMA_NSTAGE) & 1);
        R* ot = outt + (m & 1) * NF * TMA_SUB + f * TMA_SUB;

        if (m == 0) {
            // warm-up chunk: cells s0-4 .. s0+3 fill both windows; last row gives the interface s0 - 1/2
#pragma unroll
            for (int r = 0; r < TMA_CH; ++r) {
                const int c = s0 - 4 + r;
                R ud = R(0);
                if (c <= nd - 1) load_row(st, c < 0 ? r - c : r, ud);   // c < 0: row of cell 0 (outflow clamp)
                if (MODE == 2) ucell[r] = ud;
                if (r > 0) {
                    wp.push(fp_pending, c3, eps);
                    wm.push(fm2, c3, eps);
                }
                fp_pending = fp2;
            }
            R bp, np_, dp, bm, nm, dm;
            weno7_side<R, false>(wp, bp, np_, dp);
            weno7_side<R, true>(wm, bm, nm, dm);
            const R x = T::fma_(np_, dm, nm * dp) * T::rcp_(dp * dm);
            fhat_prev = T::fma_((bp + bm) + x, R(1.0 / 12.0), wp.v[0] + wm.v[0]);
            q = TMA_CH;
            if (DIR != 0 && valid) {
                if (MODE >= 1) lpre = Lf[base + (long long)s0 * stride];
                if (MODE == 2 && a.use_un) upre = Unf[base + (long long)s0 * stride];
            }
            continue;
        }
        // the U value of the emitted cell i = c - 4 was read four rows ago: keep the chunk's U column for MODE 2
#pragma unroll
        for (int r = 0; r < TMA_CH; ++r) {
            if (q + r <= len + 7) {
                const int c = s0 - 4 + q + r;
                const int i = c - 4;
                R unew = R(0);
                if (c <= nd - 1) load_row(st, r, unew);              // c > nd-1: keep the last valid split fluxes
                wp.push(fp_pending, c3, eps);
                wm.push(fm2, c3, eps);
                fp_pending = fp2;
                R bp, np_, dp, bm, nm, dm;
                weno7_side<R, false>(wp, bp, np_, dp);
                weno7_side<R, true>(wm, bm, nm, dm);
                const R x = T::fma_(np_, dm, nm * dp) * T::rcp_(dp * dm);
                const R fhat = T::fma_((bp + bm) + x, R(1.0 / 12.0), wp.v[0] + wm.v[0]);   // = 2 F_hat_{i+1/2}
                const R minus_div = (fhat_prev - fhat) * a.half_inv_dx;
                fhat_prev = fhat;
                if (DIR == 0) {
                    ot[sub_off<0>(r, lane)] = minus_div;
                } else if (valid) {
                    const long long idx = base + (long long)i * stride;
                    R lcur = lpre, ucur = upre;
                    if (i + 1 < s1) {
                        if (MODE >= 1) lpre = Lf[idx + stride];
                        if (MODE == 2 && a.use_un) upre = Unf[idx + stride];
                    }
                    if (MODE == 0) Lf[idx] = minus_div;
                    else if (MODE == 1) Lf[idx] = lcur + minus_div;
                    else {
                        // U_s of cell i: four rows behind the newest row -> previous chunk for r < 4
                        const R us = ucell[(r + 4) & 7];
                        R un = T::fma_(a.dt, lcur + minus_div, us);
                        if (a.use_un) un = T::fma_(a.rk_b, un, a.rk_a * ucur);
                        Uof[idx] = un;
                    }
                }
                if (MODE == 2) ucell[r] = unew;
            }
        }
        q += TMA_CH;
    }
    if (DIR == 0) {
        fence_proxy_async();
        if (leader) tma_wait_read0();
        __syncthreads();
        if (leader && nchunks > 1) {
            const R* src = outt + ((nchunks - 1) & 1) * NF * TMA_SUB;
            tma_store_4d(&maps.Lst, src, s0 + (nchunks - 2) * TMA_CH, t0, tfix, 0);
            tma_commit();
            tma_wait_all0();
        }
    }
}

}  // namespace hydro_dev
