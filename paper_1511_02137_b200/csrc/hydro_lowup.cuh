// hydro_lowup.cuh -- first-order update U^L of the positivity-preserving limiter (reading R16), fp64.  PRODUCT.
//
//   U^L_c = U_c - (dt/dx) sum_d (F^L_{c+1/2} - F^L_{c-1/2}),   F^L = f+_i + f-_{i+1} the first-order Lax-Friedrichs flux
//         = U_c - (dt/dx) sum_d { [ (F^d - alpha_d U)_{c+1} - (F^d + alpha_d U)_{c-1} ] / 2 + alpha_d U_c }
// with the physical fluxes of a-3 (eq. 1) and zero-gradient ghosts (a-7: a neighbour outside the grid is
// the cell itself).  A 7-point stencil over (U[NF], W, P): HBM-bound (reads NF + 2 fields, writes NF).
//
// Block = a tile of 32 x 8 columns marching along z (grid: x tiles, y tiles, z segments).  Every plane of the tile arrives
// WITH its one-cell rim as three TMA boxes (U: 36 x 10 x 1 x NF; W, P: 36 x 10 x 1 x 1) in a 3-stage shared-memory ring,
// two planes ahead of the arithmetic and signalled by mbarriers, so that no thread computes a global load address or
// waits on a global load: the in-plane neighbours are shared-memory loads at immediate offsets, the z neighbours stay in
// registers (below / here / above).  The rim cells that fall outside the grid are zero-filled by TMA and overwritten in
// shared memory with the edge cell (tiles on a grid face only; block-uniform tests).  The boxes start at x0 - 2, not x0 - 1:
// a tiled TMA load whose innermost coordinate is not a multiple of 16 bytes (an odd fp64 index) faults with "illegal
// instruction" on sm_100a (measured: boxes at x = -1, 1, 31 fault, at -2, 0 they load), so column 0 and 35 are unused.
// The direct-load kernel this replaces spent 217 non-FP64 warp-instructions per cell (64-bit address arithmetic of 30
// global loads) and 7 of 10 cycles per issued instruction on the long scoreboard (profiles/r2_ncu_kernels.md).
#pragma once
#include "hydro_sweep_ring.cuh"

namespace hydro_dev {

constexpr int LOW_BX = 32, LOW_BY = 8;                         // tile of columns per block
constexpr int LOW_TW = LOW_BX + 4, LOW_TH = LOW_BY + 2;        // with the rim; x: two cells per side, see below
constexpr int LOW_TILE = LOW_TW * LOW_TH;                      // reals per field tile (dense TMA box, x fastest)
constexpr int LOW_NST = 3;                                     // ring depth: in-plane tile, the plane above, one in flight
__host__ __device__ constexpr int low_round128(int b) { return (b + 127) / 128 * 128; }
__host__ __device__ constexpr int low_u_bytes(int nf) { return low_round128(nf * LOW_TILE * 8); }
__host__ __device__ constexpr int low_stage_bytes(int nf) { return low_u_bytes(nf) + 2 * low_round128(LOW_TILE * 8); }
__host__ __device__ constexpr int low_smem_bytes(int nf) { return LOW_NST * low_stage_bytes(nf) + 64; }
__host__ __device__ constexpr int low_blocks_per_sm(int nf) { return nf == 4 ? 4 : 3; }

struct LowMaps { CUtensorMap U, W, P; };                      // boxes (36, 10, 1, NF) and (36, 10, 1, 1) of the local array

template <int NF>
__global__ void __launch_bounds__(LOW_BX * LOW_BY, low_blocks_per_sm(NF))
k_lowup_tma(const __grid_constant__ LowMaps maps, const LowArgs<double> a, const int seg_len) {
    typedef double R;
    extern __shared__ __align__(1024) unsigned char smem[];
    constexpr int SB = low_stage_bytes(NF), UB = low_u_bytes(NF), WB = low_round128(LOW_TILE * 8);
    constexpr uint32_t TX_BYTES = (NF + 2) * LOW_TILE * 8;     // what the three boxes deliver (zero fill included)
    uint64_t* full = (uint64_t*)(smem + LOW_NST * SB);
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * LOW_BX + tx;
    const int x0 = blockIdx.x * LOW_BX, y0 = blockIdx.y * LOW_BY;
    const int k0 = blockIdx.z * seg_len, k1 = min(a.nz, k0 + seg_len);
    if (k0 >= k1) return;                                      // whole block
    const int kb = k0 > 0 ? k0 - 1 : 0, ke = min(k1, a.nz - 1);   // planes this block reads: tile n holds plane kb + n
    const int np = ke - kb + 1;

    // array t (0..NF-1: U fields, NF: W, NF+1: P) of stage s
    auto arr = [&](int s, int t) -> R* {
        return (R*)(smem + s * SB + (t < NF ? t * LOW_TILE * 8 : UB + (t - NF) * WB));
    };
    auto issue = [&](int n) {                                  // thread 0 only
        const int s = n % LOW_NST;
        mbar_expect_tx(&full[s], TX_BYTES);
        tma_load_4d(smem + s * SB, &maps.U, &full[s], x0 - 2, y0 - 1, kb + n, 0);
        tma_load_4d(smem + s * SB + UB, &maps.W, &full[s], x0 - 2, y0 - 1, kb + n, 0);
        tma_load_4d(smem + s * SB + UB + WB, &maps.P, &full[s], x0 - 2, y0 - 1, kb + n, 0);
    };
    // a-7 in the plane: rim cells outside the grid take the edge cell (the grid may end inside the tile)
    const bool fix_l = x0 == 0, fix_r = x0 + LOW_BX >= a.nx, fix_b = y0 == 0, fix_t = y0 + LOW_BY >= a.ny;
    const int cx = a.nx - x0 + 1, cy = a.ny - y0;              // tile column / row of the last cell inside the grid (cell i sits in column i - x0 + 2)
    auto fix_rim = [&](int s) {
        if (fix_l | fix_r) {
            for (int e = tid; e < (NF + 2) * LOW_BY; e += LOW_BX * LOW_BY) {
                R* t = arr(s, e / LOW_BY) + (e % LOW_BY + 1) * LOW_TW;
                if (fix_l) t[1] = t[2];
                if (fix_r) t[cx + 1] = t[cx];
            }
        }
        if (fix_b | fix_t) {
            for (int e = tid; e < (NF + 2) * LOW_BX; e += LOW_BX * LOW_BY) {
                R* t = arr(s, e / LOW_BX) + (e % LOW_BX + 2);
                if (fix_b) t[0] = t[LOW_TW];
                if (fix_t) t[(cy + 1) * LOW_TW] = t[cy * LOW_TW];
            }
        }
    };

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < LOW_NST; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int n0 = k0 - kb;                                    // tile of the first output plane (0 or 1)
    if (tid == 0)
        for (int n = 0; n <= n0 + 1 && n < np; ++n) issue(n);

    R alpha[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) alpha[d] = Real<R>::from_bits(a.diag->slot[a.slot].alpha_bits[d]);
    const int own = (ty + 1) * LOW_TW + tx + 2;                // this thread's cell inside a field tile
    auto load_cell = [&](int s, int off, LowCell<R, NF>& c) {
        const R* u = (const R*)(smem + s * SB) + off;
#pragma unroll
        for (int q = 0; q < NF; ++q) c.u[q] = u[q * LOW_TILE];
        c.w = ((const R*)(smem + s * SB + UB))[off];
        c.p = ((const R*)(smem + s * SB + UB + WB))[off];
    };

    LowCell<R, NF> below, here, above, nb;
    mbar_wait(&full[0], 0);
    if (n0 == 1) {
        load_cell(0, own, below);
        mbar_wait(&full[1], 0);
        load_cell(1, own, here);
        fix_rim(1);
    } else {
        load_cell(0, own, here);
        below = here;
        fix_rim(0);
    }
    const int i = x0 + tx, j = y0 + ty;
    const bool active = i < a.nx && j < a.ny;
    long long c = ((long long)k0 * a.ny + j) * a.nxp + i;
    const long long sz = (long long)a.nxp * a.ny;
    for (int k = k0; k < k1; ++k, c += sz) {
        const int n = k - kb, s = n % LOW_NST;
        fence_proxy_async();                                   // rim writes of tile n-1 before the TMA load that replaces it
        __syncthreads();                                       // iteration k-1 is over: tile n-1 is free, tile n's rim is fixed
        if (tid == 0 && n + 2 < np) issue(n + 2);
        if (k < a.nz - 1) {
            const int s1 = (n + 1) % LOW_NST;
            mbar_wait(&full[s1], ((n + 1) / LOW_NST) & 1);
            load_cell(s1, own, above);
            fix_rim(s1);                                       // for the next iteration; nobody reads this rim before the barrier
        } else above = here;
        R acc[NF];
        // sum over the two faces of a direction: (F^L_+ - F^L_-) = [ (F_p - alpha U_p) - (F_m + alpha U_m) ] / 2 + alpha U_c
#pragma unroll
        for (int q = 0; q < NF; ++q)
            acc[q] = R(0.5) * (low_term<R, NF>(above, 2, q, alpha[2]) - low_term<R, NF>(below, 2, q, -alpha[2])) + alpha[2] * here.u[q];
        load_cell(s, own + 1, nb);
#pragma unroll
        for (int q = 0; q < NF; ++q) acc[q] += R(0.5) * low_term<R, NF>(nb, 0, q, alpha[0]) + alpha[0] * here.u[q];
        load_cell(s, own - 1, nb);
#pragma unroll
        for (int q = 0; q < NF; ++q) acc[q] -= R(0.5) * low_term<R, NF>(nb, 0, q, -alpha[0]);
        load_cell(s, own + LOW_TW, nb);
#pragma unroll
        for (int q = 0; q < NF; ++q) acc[q] += R(0.5) * low_term<R, NF>(nb, 1, q, alpha[1]) + alpha[1] * here.u[q];
        load_cell(s, own - LOW_TW, nb);
#pragma unroll
        for (int q = 0; q < NF; ++q) acc[q] -= R(0.5) * low_term<R, NF>(nb, 1, q, -alpha[1]);
        if (active) {
#pragma unroll
            for (int q = 0; q < NF; ++q) a.UL[q * a.Np + c] = fma(-a.lam, acc[q], here.u[q]);
        }
        below = here;
        here = above;
    }
}

}  // namespace hydro_dev
