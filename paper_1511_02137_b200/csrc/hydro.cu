// hydro.cu -- C-ABI entry points of include/hydro.h: handle, buffers, launch sequence.  PRODUCT (sm_100a).
// No CPU fallback: every step of the path runs in the kernels of hydro_kernels.cuh.
#include "../../include/hydro.h"
#include "hydro_kernels.cuh"
#include "hydro_sweep_ring.cuh"
#include "hydro_lowup.cuh"

#include <cudaTypedefs.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace hydro_dev;

struct EvSpan { int cls; cudaEvent_t a, b; bool owns_a; };   // one profiled launch: [a, b] on the handle's stream
struct hydro {
    int nx, ny, nz, nf, prec, order;    // order: 7 (WENO7, the paper's scheme) or 5 (its WENO5 variant)
    int nxp;                            // row pitch in reals: nx rounded up so that a row is a multiple of 16 bytes (TMA)
    long long N, Np;                    // interior cells; field stride nxp*ny*nz
    double dx, dt, weno_eps, delta, e_floor;
    double sigma;                       // Gaussian deposit width [fm]; 0 = point deposit
    int limiter;                        // 1: positivity-preserving flux limiter (R16; fp64 only)
    bool tail_split;                    // sweeps: short blocks for the partial last wave (HYDRO_NO_TAIL_SPLIT=1 disables)
    int nz_global, k_offset, own_lo, own_hi;   // z-slab decomposition (f-4); defaults: nz, 0, 0, nz
    size_t esz;                         // bytes per real
    cudaStream_t stream;
    bool own_stream;
    void* buf[3];                       // state copies: buf[cur] = U^n, the other two are stage states
    int cur;
    void* L;                            // right-hand side
    void* P;                            // pressure of the state the primitives were last computed for
    void* W;                            // scale/(E+p) of that state
    Diag* diag;
    JetDev* jets_dev;
    std::vector<JetDev> jets;
    bool jets_dirty;
    long long step;
    int prim_slot;                      // DiagSlot holding alpha of buf[cur]'s primitives
    bool prims_valid;
    // ring sweeps: tensor maps per buffer (0..2 state copies, 3 = L) and direction, march cells per block
    CUtensorMap mapB[4][3], mapW[3], mapP[3];
    // nf = 5 in fp64 without the limiter: fields 0..3 by the 4-warp kernel (boxes of 4 of the 5 fields) + the baryon
    // density by the one-warp kernel (boxes of 1 field)
    CUtensorMap mapB4[4][3], mapB1[4][3], vmapB4[4][3], vmapB1[4][3];
    bool split5;                        // HYDRO_NO_SPLIT5=1 keeps the 5-warp kernel
    // z-slab decomposition: the same maps over the OWNED planes only (x/y sweeps of the owned planes while the halos are
    // still in flight; output clipping of the z sweep); built by hydro_set_slab
    CUtensorMap vmapB[4][3], vmapW[3], vmapP[3];
    bool view;                          // launch the sweeps on the owned-planes view (hydro_stage_sweeps_part)
    CUtensorMap mapLowB[3], mapLowW, mapLowP;   // limiter (fp64): plane tiles with their rim for k_lowup_tma (hydro_lowup.cuh)
    int seg_len[3], tma_nseg[3];
    int num_sms;
    int prim_blocks_per_sm;             // resident k_prim blocks per SM (occupancy query at create)
    long long launches;
    // one RK3 step captured as a CUDA graph (replayed by hydro_step when profiling is off): valid for graph_slot only and
    // until the jets, the limiter, the deposit width or the slab change
    cudaGraphExec_t graph;
    int graph_slot, graph_njets;
    long long graph_launches;           // kernel launches inside the graph
    bool use_graph;                     // HYDRO_NO_GRAPH=1 disables
    // profiling
    bool profiling;
    std::vector<EvSpan> ev_inflight;
    std::vector<cudaEvent_t> ev_pool;
    cudaEvent_t chain_prev;             // end event of the previous profiled launch (0: start a new chain)
    double k_ms[HYDRO_K_COUNT];
    long long k_n[HYDRO_K_COUNT];
    std::string cuda_err;
};

namespace {

int cuda_fail(hydro* h, cudaError_t e, const char* where) {
    if (h) {
        char b[256];
        snprintf(b, sizeof b, "%s: %s", where, cudaGetErrorString(e));
        h->cuda_err = b;
    }
    return e == cudaErrorMemoryAllocation ? HYDRO_ENOMEM : HYDRO_ECUDA;
}
#define CK(call)                                                        \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);          \
    } while (0)

// Per-launch device times when profiling is on: ONE event after every launch; a launch's start is the previous
// launch's end event (launches of a step are back to back on the stream), so profiling costs one event per launch.
cudaEvent_t get_event(hydro* h) {
    cudaEvent_t e = 0;
    if (!h->ev_pool.empty()) { e = h->ev_pool.back(); h->ev_pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}
struct Timer {
    hydro* h;
    EvSpan sp;
    bool on;
    Timer(hydro* h_, int cls_) : h(h_), on(h_->profiling) {
        if (!on) return;
        sp.cls = cls_;
        if (h->chain_prev) { sp.a = h->chain_prev; sp.owns_a = false; }
        else { sp.a = get_event(h); sp.owns_a = true; cudaEventRecord(sp.a, h->stream); }
    }
    ~Timer() {
        if (!on) return;
        sp.b = get_event(h);
        cudaEventRecord(sp.b, h->stream);
        h->ev_inflight.push_back(sp);
        h->chain_prev = sp.b;
    }
};

void drain_events(hydro* h) {
    for (size_t n = 0; n < h->ev_inflight.size(); ++n) {
        const EvSpan& sp = h->ev_inflight[n];
        float ms = 0.f;
        cudaEventSynchronize(sp.b);
        cudaEventElapsedTime(&ms, sp.a, sp.b);
        h->k_ms[sp.cls] += ms;
        h->k_n[sp.cls] += 1;
    }
    for (size_t n = 0; n < h->ev_inflight.size(); ++n) {
        if (h->ev_inflight[n].owns_a) h->ev_pool.push_back(h->ev_inflight[n].a);
        h->ev_pool.push_back(h->ev_inflight[n].b);
    }
    h->ev_inflight.clear();
    h->chain_prev = 0;
}

// con2prim (+ wavespeed maxima if with_alpha) of the z planes [k0, k1); reset: clear the DiagSlot first
template <typename R>
int launch_prim_range(hydro* h, const void* U, int slot, int k0, int k1, bool reset, bool with_alpha) {
    if (reset) CK(cudaMemsetAsync(&h->diag->slot[slot], 0, sizeof(DiagSlot), h->stream));
    if (k1 <= k0) return HYDRO_OK;
    const long long plane = (long long)h->nx * h->ny;
    PrimArgs<R> a;
    a.U = (const R*)U; a.P = (R*)h->P; a.W = (R*)h->W; a.diag = h->diag; a.slot = slot; a.c0 = k0 * plane; a.N = k1 * plane;
    a.Np = h->Np; a.nx = h->nx; a.nxp = h->nxp; a.with_alpha = with_alpha ? 1 : 0;
    a.seed_slot = (slot + NSLOT - 1) % NSLOT;                       // the previous stage's slot: its arg[] names good candidates
    a.own_lo = (long long)h->own_lo * plane; a.own_hi = (long long)h->own_hi * plane;
    a.e_floor = (R)h->e_floor; a.one_minus_delta = (R)(1.0 - h->delta);
    // grid-stride over the range with exactly one wave of resident blocks (no partial last wave)
    long long blocks = (a.N - a.c0 + PRIM_THREADS - 1) / PRIM_THREADS;
    long long cap = (long long)h->num_sms * h->prim_blocks_per_sm;
    if (blocks > cap) blocks = cap;
    {
        Timer t(h, HYDRO_K_PRIM);
        k_prim<R><<<(unsigned)blocks, PRIM_THREADS, 0, h->stream>>>(a);
    }
    h->launches += 1;
    CK(cudaGetLastError());
    return HYDRO_OK;
}
template <typename R>
int launch_prim(hydro* h, const void* U, int slot) { return launch_prim_range<R>(h, U, slot, 0, h->nz, true, true); }

// 0..2: the state copies, 3: the RHS buffer L
int buf_index(const hydro* h, const void* U) {
    for (int b = 0; b < 3; ++b) if (h->buf[b] == U) return b;
    return U == h->L ? 3 : -1;
}

// One ring sweep (hydro_sweep_ring.cuh).  `Us` must be one of the three state buffers; `out_b` is the buffer (0..2 state
// copy, 3 = L) the result is stored / reduced into; `un_b` that of U^n (OUT_COMBINE; < 0: none).
// LIM = 1 (fp64 only): the limited scheme of R16, U^L is read from h->L.
// h->view (z-slabs): the x and y sweeps run on the owned planes only (all maps are the owned-planes views, the kernel
// sees a grid of own_hi - own_lo planes); the z sweep marches the whole local array as always (what it adds to the halo
// planes of the target is overwritten by the next exchange).
template <typename R, int ORDER, int LIM, int DIR, int OUT, int NF>
int launch_ring_nf(hydro* h, const void* Us, int slot, int out_b, int un_b, double coef, double rk_a, double rk_b) {
    if constexpr (LIM && sizeof(R) != 8) return HYDRO_ESTATE;
    else {
        const int b = buf_index(h, Us);
        if (b < 0 || b > 2 || out_b < 0 || out_b > 3 || un_b > 2) return HYDRO_ESTATE;
        const bool vw = h->view && DIR != 2;                               // everything through the owned-planes view
        // which box the maps carry: all nf fields, or (5-field state split over two kernels) 4 fields / 1 field
        CUtensorMap (*mB)[3] = NF == h->nf ? h->mapB : NF == 4 ? h->mapB4 : h->mapB1;
        CUtensorMap (*vB)[3] = NF == h->nf ? h->vmapB : NF == 4 ? h->vmapB4 : h->vmapB1;
        RingMaps m;
        m.U = vw ? vB[b][DIR] : mB[b][DIR];
        m.W = vw ? h->vmapW[DIR] : h->mapW[DIR];
        m.P = vw ? h->vmapP[DIR] : h->mapP[DIR];
        m.Out = vw ? vB[out_b][DIR] : mB[out_b][DIR];
        m.Un = un_b >= 0 ? (vw ? vB[un_b][DIR] : mB[un_b][DIR]) : m.Out;
        m.UL = vw ? vB[3][DIR] : mB[3][DIR];
        const int nz_k = vw ? h->own_hi - h->own_lo : h->nz;              // planes the kernel sees
        RingArgs a;
        a.diag = h->diag; a.slot = slot; a.nx = h->nx; a.ny = h->ny; a.nz = nz_k; a.seg_len = h->seg_len[DIR];
        a.eps_eff = (ORDER == 5 ? 48.0 : 144.0 / 39.0) * h->weno_eps; a.coef = coef; a.dt = h->dt; a.rk_a = rk_a; a.rk_b = rk_b;
        a.k3lam = 3.0 * h->dt / h->dx / (ORDER == 5 ? 6.0 : 12.0); a.nlim = &h->diag->nlim_total;
        a.own_lo = vw ? 0 : h->own_lo; a.own_hi = vw ? nz_k : h->own_hi;
        const int nlane = DIR == 0 ? h->ny : h->nx;
        const int other = DIR == 2 ? h->ny : nz_k;
        const int nd = DIR == 0 ? h->nx : DIR == 1 ? h->ny : h->nz;
        const long long tiles = (long long)((nlane + 31) / 32) * other;
        dim3 grid((unsigned)tiles, (unsigned)h->tma_nseg[DIR], 1);
        a.n_long = -1; a.short_nseg = 1; a.short_len = nd;
        // tail splitting: whole-line blocks for the complete waves, short blocks for the partial last wave
        const long long slots = (long long)h->num_sms * ring_blocks_per_sm(NF, sizeof(R), OUT, LIM);
        if (h->tail_split && h->tma_nseg[DIR] == 1 && tiles > slots && tiles % slots != 0 && nd >= 64) {
            const long long n_long = tiles / slots * slots, rem = tiles - n_long;
            int best_k = 1;
            double best = 1.0;                                          // cost of the last wave in units of a whole-line wave
            for (int k = 2; k <= 8 && nd / k >= 32; k *= 2) {
                const int sl = ((nd + k - 1) / k + RING_CH - 1) / RING_CH * RING_CH;
                const int kk = (nd + sl - 1) / sl;
                const double waves = (double)((rem * kk + slots - 1) / slots);
                const double cost = waves * (sl + RING_CH) / (double)(nd + RING_CH);
                if (cost < best - 1e-9) { best = cost; best_k = kk; a.short_len = sl; }
            }
            if (best_k > 1) {
                a.n_long = (int)n_long; a.short_nseg = best_k;
                grid = dim3((unsigned)(n_long + rem * best_k), 1, 1);
            } else a.short_len = nd;
        }
        dim3 block(32, NF, 1);
        {
            Timer t(h, HYDRO_K_SWEEP_X + DIR);
            k_sweep_ring<R, ORDER, LIM, DIR, OUT, NF><<<grid, block, ring_smem_bytes(NF, OUT, sizeof(R), LIM), h->stream>>>(m, a);
        }
        h->launches += 1;
        CK(cudaGetLastError());
        return HYDRO_OK;
    }
}

template <typename R, int LIM, int DIR, int OUT>
int launch_ring_lim(hydro* h, const void* Us, int slot, int out_b, int un_b, double coef, double rk_a, double rk_b) {
    if constexpr (!LIM && sizeof(R) == 8) {
        if (h->nf == 5 && h->split5) {
            int rc = h->order == 5 ? launch_ring_nf<R, 5, 0, DIR, OUT, 4>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b)
                                   : launch_ring_nf<R, 7, 0, DIR, OUT, 4>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b);
            if (rc != HYDRO_OK) return rc;
            return h->order == 5 ? launch_ring_nf<R, 5, 0, DIR, OUT, 1>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b)
                                 : launch_ring_nf<R, 7, 0, DIR, OUT, 1>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b);
        }
    }
    if (h->order == 5)
        return h->nf == 4 ? launch_ring_nf<R, 5, LIM, DIR, OUT, 4>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b)
                          : launch_ring_nf<R, 5, LIM, DIR, OUT, 5>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b);
    return h->nf == 4 ? launch_ring_nf<R, 7, LIM, DIR, OUT, 4>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b)
                      : launch_ring_nf<R, 7, LIM, DIR, OUT, 5>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b);
}
template <typename R, int DIR, int OUT>
int launch_ring(hydro* h, const void* Us, int slot, int out_b, int un_b, double coef, double rk_a, double rk_b) {
    return h->limiter ? launch_ring_lim<R, 1, DIR, OUT>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b)
                      : launch_ring_lim<R, 0, DIR, OUT>(h, Us, slot, out_b, un_b, coef, rk_a, rk_b);
}

template <typename R, int LIM, int DIR, int OUT, int NF>
int set_smem_attr() {
    if constexpr (LIM && sizeof(R) != 8) return 0;
    else
        return (cudaFuncSetAttribute(k_sweep_ring<R, 7, LIM, DIR, OUT, NF>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     ring_smem_bytes(NF, OUT, sizeof(R), LIM)) == cudaSuccess ? 0 : 1) +
               (cudaFuncSetAttribute(k_sweep_ring<R, 5, LIM, DIR, OUT, NF>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     ring_smem_bytes(NF, OUT, sizeof(R), LIM)) == cudaSuccess ? 0 : 1);
}
template <typename R>
int set_smem_attrs_baryon() {
    if constexpr (sizeof(R) != 8) return 0;
    else return set_smem_attr<R, 0, 0, OUT_STORE, 1>() + set_smem_attr<R, 0, 0, OUT_COMBINE1, 1>() +
                set_smem_attr<R, 0, 0, OUT_COMBINE, 1>() + set_smem_attr<R, 0, 1, OUT_REDUCE, 1>() +
                set_smem_attr<R, 0, 2, OUT_REDUCE, 1>();
}
template <typename R, int NF>
int set_smem_attrs() {
    return set_smem_attr<R, 0, 0, OUT_STORE, NF>() + set_smem_attr<R, 0, 0, OUT_COMBINE1, NF>() +
           set_smem_attr<R, 0, 0, OUT_COMBINE, NF>() + set_smem_attr<R, 0, 1, OUT_REDUCE, NF>() +
           set_smem_attr<R, 0, 2, OUT_REDUCE, NF>() + set_smem_attr<R, 1, 0, OUT_COMBINE1, NF>() +
           set_smem_attr<R, 1, 0, OUT_COMBINE, NF>() + set_smem_attr<R, 1, 1, OUT_REDUCE, NF>() +
           set_smem_attr<R, 1, 2, OUT_REDUCE, NF>();
}

// 4-D tensor map (x, y, z, field) of the z planes [k0, k1) of one SoA buffer with `nfb` fields; box given per dimension
int make_map(hydro* h, CUtensorMap* out, void* base0, int nfb, const unsigned box[4], bool swizzle64, int k0, int k1) {
    void* base = (char*)base0 + (size_t)k0 * h->nxp * h->ny * h->esz;
    static PFN_cuTensorMapEncodeTiled_v12000 encode = 0;
    if (!encode) {
        void* fn = 0;
        cudaDriverEntryPointQueryResult q;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
        if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) {
            h->cuda_err = "cuTensorMapEncodeTiled entry point not available";
            return HYDRO_ECUDA;
        }
        encode = (PFN_cuTensorMapEncodeTiled_v12000)fn;
    }
    cuuint64_t gdim[4] = {(cuuint64_t)h->nx, (cuuint64_t)h->ny, (cuuint64_t)(k1 - k0), (cuuint64_t)nfb};
    const cuuint64_t es8 = (cuuint64_t)h->esz;
    cuuint64_t gstr[3] = {(cuuint64_t)h->nxp * es8, (cuuint64_t)h->nxp * h->ny * es8, (cuuint64_t)h->Np * es8};
    cuuint32_t bx[4] = {box[0], box[1], box[2], box[3]};
    cuuint32_t es[4] = {1, 1, 1, 1};
    // x sweep boxes (8 cells of x innermost = 64 bytes in fp64, 32 bytes in fp32) are swizzled at their own width
    const CUtensorMapSwizzle swz = !swizzle64 ? CU_TENSOR_MAP_SWIZZLE_NONE
                                              : (h->esz == 8 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_32B);
    CUresult r = encode(out, h->esz == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, gdim,
                        gstr, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char b[96];
        snprintf(b, sizeof b, "cuTensorMapEncodeTiled failed (%d)", (int)r);
        h->cuda_err = b;
        return HYDRO_ECUDA;
    }
    return HYDRO_OK;
}

// tensor maps of the planes [k0, k1) of every buffer, per direction; boxes of `boxf` fields (mW, mP may be null)
int build_maps(hydro* h, CUtensorMap mB[4][3], CUtensorMap mW[3], CUtensorMap mP[3], int k0, int k1, unsigned boxf) {
    const unsigned boxes[3][4] = {{RING_CH, 32, 1, boxf}, {32, RING_CH, 1, boxf}, {32, 1, RING_CH, boxf}};
    int rc;
    for (int d = 0; d < 3; ++d) {
        unsigned b1[4] = {boxes[d][0], boxes[d][1], boxes[d][2], 1};
        for (int b = 0; b < 4; ++b)
            if ((rc = make_map(h, &mB[b][d], b < 3 ? h->buf[b] : h->L, h->nf, boxes[d], d == 0, k0, k1)) != HYDRO_OK) return rc;
        if (mW && (rc = make_map(h, &mW[d], h->W, 1, b1, d == 0, k0, k1)) != HYDRO_OK) return rc;
        if (mP && (rc = make_map(h, &mP[d], h->P, 1, b1, d == 0, k0, k1)) != HYDRO_OK) return rc;
    }
    return HYDRO_OK;
}
// all map sets of the planes [k0, k1): full boxes, and the 4 + 1 split of a 5-field state
int build_map_sets(hydro* h, bool view, int k0, int k1) {
    int rc;
    if ((rc = build_maps(h, view ? h->vmapB : h->mapB, view ? h->vmapW : h->mapW, view ? h->vmapP : h->mapP, k0, k1,
                         (unsigned)h->nf)) != HYDRO_OK) return rc;
    if (h->nf == 5) {
        if ((rc = build_maps(h, view ? h->vmapB4 : h->mapB4, 0, 0, k0, k1, 4)) != HYDRO_OK) return rc;
        if ((rc = build_maps(h, view ? h->vmapB1 : h->mapB1, 0, 0, k0, k1, 1)) != HYDRO_OK) return rc;
    }
    return HYDRO_OK;
}

int setup_tma(hydro* h) {
    int rc;
    if ((rc = build_map_sets(h, false, 0, h->nz)) != HYDRO_OK) return rc;
    if ((rc = build_map_sets(h, true, 0, h->nz)) != HYDRO_OK) return rc;
    const int bad = h->prec == 64 ? (h->nf == 4 ? set_smem_attrs<double, 4>()
                                                : set_smem_attrs<double, 5>() + set_smem_attrs<double, 4>() + set_smem_attrs_baryon<double>())
                                  : (h->nf == 4 ? set_smem_attrs<float, 4>() : set_smem_attrs<float, 5>());
    if (bad) {
        h->cuda_err = "cudaFuncSetAttribute(max dynamic shared memory) failed";
        return HYDRO_ECUDA;
    }
    if (h->prec == 64) {                // the limiter's first-order update: 34 x 10 plane tiles (32 x 8 columns + rim)
        const unsigned bu[4] = {(unsigned)LOW_TW, (unsigned)LOW_TH, 1u, (unsigned)h->nf}, b1[4] = {(unsigned)LOW_TW, (unsigned)LOW_TH, 1u, 1u};
        for (int b = 0; b < 3; ++b)
            if ((rc = make_map(h, &h->mapLowB[b], h->buf[b], h->nf, bu, false, 0, h->nz)) != HYDRO_OK) return rc;
        if ((rc = make_map(h, &h->mapLowW, h->W, 1, b1, false, 0, h->nz)) != HYDRO_OK) return rc;
        if ((rc = make_map(h, &h->mapLowP, h->P, 1, b1, false, 0, h->nz)) != HYDRO_OK) return rc;
        if (cudaFuncSetAttribute(k_lowup_tma<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, low_smem_bytes(4)) != cudaSuccess ||
            cudaFuncSetAttribute(k_lowup_tma<5>, cudaFuncAttributeMaxDynamicSharedMemorySize, low_smem_bytes(5)) != cudaSuccess) {
            h->cuda_err = "cudaFuncSetAttribute(max dynamic shared memory, k_lowup_tma) failed";
            return HYDRO_ECUDA;
        }
    }
    // march segments: one per line unless the grid is too small to fill the machine; multiples of the chunk
    const int nd[3] = {h->nx, h->ny, h->nz};
    for (int d = 0; d < 3; ++d) {
        const long long nlane = d == 0 ? h->ny : h->nx;
        const long long other = d == 2 ? h->ny : h->nz;
        const long long blocks1 = ((nlane + 31) / 32) * other;
        int seg = 1;
        while (blocks1 * seg < (long long)h->num_sms * ring_blocks_per_sm(h->nf, (int)h->esz) && nd[d] / (seg * 2) >= 16) seg *= 2;
        int ls = (nd[d] + seg - 1) / seg;
        ls = (ls + RING_CH - 1) / RING_CH * RING_CH;
        const char* force = getenv("HYDRO_SEG_LEN");                  // tuning knob: march cells per block
        if (force && atoi(force) >= RING_CH) ls = atoi(force) / RING_CH * RING_CH;
        h->seg_len[d] = ls;
        h->tma_nseg[d] = (nd[d] + ls - 1) / ls;
    }
    return HYDRO_OK;
}

template <typename R>
int upload_jets(hydro* h) {
    if (!h->jets_dirty) return HYDRO_OK;
    if (!h->jets.empty())
        CK(cudaMemcpyAsync(h->jets_dev, h->jets.data(), h->jets.size() * sizeof(JetDev), cudaMemcpyHostToDevice,
                           h->stream));
    // the host vector may change before the copy runs: pageable copies are staged synchronously by the runtime
    h->jets_dirty = false;
    return HYDRO_OK;
}

template <typename R>
int launch_source(hydro* h, int slot, int stage, double stage_c, bool commit, double rk_weight, void* target, double scale,
                  bool advance = false) {
    int rc;
    if ((rc = upload_jets<R>(h)) != HYDRO_OK) return rc;
    SourceArgs s;
    s.diag = h->diag; s.jets = h->jets_dev; s.njets = (int)h->jets.size(); s.slot = slot; s.stage = stage;
    s.commit = commit ? 1 : 0; s.nx = h->nx; s.ny = h->ny; s.nz = h->nz; s.nxp = h->nxp; s.N = h->Np;
    s.zero_slot = commit ? (slot + 1) % NSLOT : -1;                 // the slot the next k_prim fills
    s.advance = advance ? 1 : 0;
    s.nz_global = h->nz_global; s.k_offset = h->k_offset; s.own_lo = h->own_lo; s.own_hi = h->own_hi;
    s.stage_c = stage_c; s.dx = h->dx; s.dt = h->dt; s.rk_weight = rk_weight; s.scale = scale; s.sigma = h->sigma;
    {
        Timer t(h, HYDRO_K_SOURCE);
        k_source<R><<<1, SOURCE_THREADS, 0, h->stream>>>(s, (const R*)h->P, (R*)target);
    }
    h->launches += 1;
    CK(cudaGetLastError());
    return HYDRO_OK;
}

// With Uout: the x sweep stores U_next = a U^n + b (U_s + dt L_x), the source kernel and the y, z sweeps add b dt S,
// b dt L_y, b dt L_z to it (the stage update is linear in L).  Without: L into h->L.
// `parts`: bit 0 = x sweep + source + y sweep, bit 1 = z sweep (3 = the whole stage; the split serves the z-slab overlap:
// x and y need no z halos).  The limiter path and hydro_eval_rhs always run whole.
template <typename R>
int eval_stage_ring(hydro* h, const void* Uin, int slot, int stage, double stage_c, bool commit, double rk_weight,
                    void* Uout, const void* Un, double rk_a, double rk_b, int parts = 3) {
    const double hid = 0.5 / h->dx;
    int rc;
    if (h->limiter) {
        if (parts != 3) return HYDRO_ESTATE;
        // R16: U^L (first-order update) into h->L, then the sweeps add only theta x (WENO correction) to it
        LowArgs<R> la;
        la.U = (const R*)Uin; la.P = (const R*)h->P; la.W = (const R*)h->W; la.UL = (R*)h->L; la.diag = h->diag; la.slot = slot;
        la.nx = h->nx; la.ny = h->ny; la.nz = h->nz; la.nxp = h->nxp; la.nf = h->nf; la.N = h->N; la.Np = h->Np;
        la.lam = (R)(h->dt / h->dx);
        {
            const long long cols = (long long)((h->nx + 31) / 32) * ((h->ny + 7) / 8);
            int segs = 1;                                               // z segments: enough blocks to fill the machine
            // (measured at 256^3, 256 columns: 2 / 4 / 8 / 16 segments -> 0.239 / 0.232 / 0.228 / 0.219 ms per launch)
            while (cols * segs < (long long)h->num_sms * 16 && h->nz / (segs * 2) >= 8) segs *= 2;
            const int seg_len = (h->nz + segs - 1) / segs;
            if ((h->ny + 7) / 8 > 65535) return HYDRO_EINVAL;
            Timer t(h, HYDRO_K_PRIM);
            const dim3 grid((unsigned)((h->nx + 31) / 32), (unsigned)((h->ny + 7) / 8), (unsigned)((h->nz + seg_len - 1) / seg_len));
            if constexpr (sizeof(R) == 8) {
                const int bi = buf_index(h, Uin);
                if (bi < 0 || bi > 2) return HYDRO_ESTATE;
                LowMaps lm;
                lm.U = h->mapLowB[bi]; lm.W = h->mapLowW; lm.P = h->mapLowP;
                if (h->nf == 4) k_lowup_tma<4><<<grid, dim3(LOW_BX, LOW_BY, 1), low_smem_bytes(4), h->stream>>>(lm, la, seg_len);
                else k_lowup_tma<5><<<grid, dim3(LOW_BX, LOW_BY, 1), low_smem_bytes(5), h->stream>>>(lm, la, seg_len);
            } else return HYDRO_ESTATE;                                    // the limiter is fp64 only (hydro_set_limiter)
        }
        h->launches += 1;
        CK(cudaGetLastError());
        if (!Uout) {
            // hydro_eval_rhs: limited Euler update into a free state buffer, L = (update - U_s) / dt into another
            void* Ue = h->buf[(h->cur + 1) % 3];
            void* Ld = h->buf[(h->cur + 2) % 3];
            const int be = buf_index(h, Ue);
            if ((rc = launch_ring<R, 0, OUT_COMBINE1>(h, Uin, slot, be, -1, hid, 0.0, 1.0)) != HYDRO_OK) return rc;
            if ((rc = launch_source<R>(h, slot, stage, stage_c, commit, rk_weight, Ue, h->dt)) != HYDRO_OK) return rc;
            if ((rc = launch_ring<R, 1, OUT_REDUCE>(h, Uin, slot, be, -1, h->dt * hid, 0.0, 0.0)) != HYDRO_OK) return rc;
            if ((rc = launch_ring<R, 2, OUT_REDUCE>(h, Uin, slot, be, -1, h->dt * hid, 0.0, 0.0)) != HYDRO_OK) return rc;
            const long long n = h->Np * h->nf;
            long long bl = (n + 255) / 256;
            if (bl > (long long)h->num_sms * 16) bl = (long long)h->num_sms * 16;
            {
                Timer t(h, HYDRO_K_PRIM);
                k_diff<R><<<(unsigned)bl, 256, 0, h->stream>>>((const R*)Ue, (const R*)Uin, (R*)Ld, n, (R)(1.0 / h->dt));
            }
            h->launches += 1;
            CK(cudaGetLastError());
            return HYDRO_OK;
        }
    }
    if (Uout) {
        const int bo = buf_index(h, Uout), bn = Un ? buf_index(h, Un) : -1;
        if (bo < 0 || bo > 2 || (Un && (bn < 0 || bn > 2))) return HYDRO_ESTATE;
        const double bdt = (Un ? rk_b : 1.0) * h->dt;
        if (parts & 1) {
            if (Un) rc = launch_ring<R, 0, OUT_COMBINE>(h, Uin, slot, bo, bn, hid, rk_a, rk_b);
            else rc = launch_ring<R, 0, OUT_COMBINE1>(h, Uin, slot, bo, -1, hid, 0.0, 1.0);
            if (rc != HYDRO_OK) return rc;
            if ((rc = launch_source<R>(h, slot, stage, stage_c, commit, rk_weight, Uout, bdt, commit && stage == 2)) != HYDRO_OK) return rc;
            if ((rc = launch_ring<R, 1, OUT_REDUCE>(h, Uin, slot, bo, -1, bdt * hid, 0.0, 0.0)) != HYDRO_OK) return rc;
        }
        if (parts & 2) return launch_ring<R, 2, OUT_REDUCE>(h, Uin, slot, bo, -1, bdt * hid, 0.0, 0.0);
        return HYDRO_OK;
    }
    if (parts != 3) return HYDRO_ESTATE;
    if ((rc = launch_ring<R, 0, OUT_STORE>(h, Uin, slot, 3, -1, hid, 0.0, 0.0)) != HYDRO_OK) return rc;
    if ((rc = launch_source<R>(h, slot, stage, stage_c, commit, rk_weight, h->L, 1.0)) != HYDRO_OK) return rc;
    if ((rc = launch_ring<R, 1, OUT_REDUCE>(h, Uin, slot, 3, -1, hid, 0.0, 0.0)) != HYDRO_OK) return rc;
    return launch_ring<R, 2, OUT_REDUCE>(h, Uin, slot, 3, -1, hid, 0.0, 0.0);
}

// L(U_in, t_n + stage_c dt) into h->L; if Uout != 0 the stage combination forms the next stage state instead.
template <typename R>
int eval_stage(hydro* h, const void* Uin, int slot, int stage, double stage_c, bool commit, double rk_weight,
               void* Uout, const void* Un, double rk_a, double rk_b, int parts = 3) {
    return eval_stage_ring<R>(h, Uin, slot, stage, stage_c, commit, rk_weight, Uout, Un, rk_a, rk_b, parts);
}

template <typename R>
int ensure_prims(hydro* h) {
    if (h->prims_valid) return HYDRO_OK;
    int rc = launch_prim<R>(h, h->buf[h->cur], h->prim_slot);
    if (rc == HYDRO_OK) h->prims_valid = true;
    return rc;
}

// One RK3 step: 15 kernels.  The DiagSlots rotate slot0 -> slot0+1 -> slot0+2 -> slot0 (mod 3), so every step uses the same
// sequence; nothing the kernels are passed changes from step to step (the step counter lives in diag->step), which is
// what lets one captured step be replayed.  k_source clears the slot of the following k_prim (no memset nodes).
template <typename R>
int enqueue_step(hydro* h) {
    int rc;
    void* Un = h->buf[h->cur];
    void* Ua = h->buf[(h->cur + 1) % 3];
    void* Ub = h->buf[(h->cur + 2) % 3];
    const int s0 = h->prim_slot, s1 = (s0 + 1) % NSLOT, s2 = (s0 + 2) % NSLOT;
    // stage 1: U1 = Un + dt L(Un, t_n)
    if ((rc = eval_stage<R>(h, Un, s0, 0, 0.0, true, 1.0 / 6.0, Ua, 0, 0.0, 1.0)) != HYDRO_OK) return rc;
    if ((rc = launch_prim_range<R>(h, Ua, s1, 0, h->nz, false, true)) != HYDRO_OK) return rc;
    // stage 2: U2 = 3/4 Un + 1/4 (U1 + dt L(U1, t_n + dt))
    if ((rc = eval_stage<R>(h, Ua, s1, 1, 1.0, true, 1.0 / 6.0, Ub, Un, 0.75, 0.25)) != HYDRO_OK) return rc;
    if ((rc = launch_prim_range<R>(h, Ub, s2, 0, h->nz, false, true)) != HYDRO_OK) return rc;
    // stage 3: U^{n+1} = 1/3 Un + 2/3 (U2 + dt L(U2, t_n + dt/2)), written over Un (each cell reads only its own Un)
    if ((rc = eval_stage<R>(h, Ub, s2, 2, 0.5, true, 2.0 / 3.0, Un, Un, 1.0 / 3.0, 2.0 / 3.0)) != HYDRO_OK) return rc;
    return launch_prim_range<R>(h, Un, s0, 0, h->nz, false, true);
}

void drop_graph(hydro* h) {
    if (h->graph) cudaGraphExecDestroy(h->graph);
    h->graph = 0;
}

template <typename R>
int capture_step(hydro* h) {
    int rc;
    if ((rc = upload_jets<R>(h)) != HYDRO_OK) return rc;            // host -> device copies cannot be captured
    const long long l0 = h->launches;
    cudaGraph_t g = 0;
    CK(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
    rc = enqueue_step<R>(h);
    cudaError_t e = cudaStreamEndCapture(h->stream, &g);
    h->graph_launches = h->launches - l0;
    h->launches = l0;                                               // nothing ran yet
    if (rc != HYDRO_OK) { if (g) cudaGraphDestroy(g); return rc; }
    if (e != cudaSuccess) return cuda_fail(h, e, "cudaStreamEndCapture");
    e = cudaGraphInstantiate(&h->graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { h->graph = 0; return cuda_fail(h, e, "cudaGraphInstantiate"); }
    h->graph_slot = h->prim_slot;
    h->graph_njets = (int)h->jets.size();
    return HYDRO_OK;
}

template <typename R>
int step_impl(hydro* h, int nsteps) {
    int rc;
    if (nsteps == 0) return HYDRO_OK;
    if ((rc = ensure_prims<R>(h)) != HYDRO_OK) return rc;
    const bool graph = h->use_graph && !h->profiling;              // per-kernel event timing needs individual launches
    if (graph) {
        if ((rc = upload_jets<R>(h)) != HYDRO_OK) return rc;       // the jet table itself lives in device memory
        if (!h->graph || h->graph_njets != (int)h->jets.size() || h->graph_slot != h->prim_slot) {
            drop_graph(h);
            if ((rc = capture_step<R>(h)) != HYDRO_OK) return rc;
        }
    }
    for (int n = 0; n < nsteps; ++n) {
        if (graph) {
            CK(cudaGraphLaunch(h->graph, h->stream));
            h->launches += h->graph_launches;
        } else if ((rc = enqueue_step<R>(h)) != HYDRO_OK) return rc;
        h->step += 1;
    }
    return HYDRO_OK;
}

// ---- stage-level stepping (z-slab decomposition, f-4): the caller exchanges alpha / halos between the calls
struct StagePlan { void* in; void* out; const void* un; int slot; double c, w, a, b; };
StagePlan stage_plan(hydro* h, int s) {
    void* Un = h->buf[h->cur];
    void* Ua = h->buf[(h->cur + 1) % 3];
    void* Ub = h->buf[(h->cur + 2) % 3];
    const int slot = h->prim_slot;
    StagePlan p;
    if (s == 0) { p.in = Un; p.out = Ua; p.un = 0; p.slot = slot; p.c = 0.0; p.w = 1.0 / 6.0; p.a = 0.0; p.b = 1.0; }
    else if (s == 1) { p.in = Ua; p.out = Ub; p.un = Un; p.slot = (slot + 1) % NSLOT; p.c = 1.0; p.w = 1.0 / 6.0; p.a = 0.75; p.b = 0.25; }
    else { p.in = Ub; p.out = Un; p.un = Un; p.slot = (slot + 2) % NSLOT; p.c = 0.5; p.w = 2.0 / 3.0; p.a = 1.0 / 3.0; p.b = 2.0 / 3.0; }
    return p;
}
// part: -1 = all planes; 0 = the owned planes (+ the local wavespeed maxima and cap counts); 1 = the halo planes
// (primitives only), to be called once the neighbours' planes have been unpacked
template <typename R>
int stage_prims_impl(hydro* h, int s, int part) {
    const StagePlan p = stage_plan(h, s);
    if (part < 0) return launch_prim<R>(h, p.in, p.slot);
    if (part == 0) return launch_prim_range<R>(h, p.in, p.slot, h->own_lo, h->own_hi, true, true);
    int rc = launch_prim_range<R>(h, p.in, p.slot, 0, h->own_lo, false, false);
    if (rc != HYDRO_OK) return rc;
    return launch_prim_range<R>(h, p.in, p.slot, h->own_hi, h->nz, false, false);
}
// part: -1 = the whole stage on the whole local array; 0 = x sweep + source + y sweep on the owned planes;
// 1 = z sweep and, for s = 2, the end-of-step bookkeeping
template <typename R>
int stage_sweeps_impl(hydro* h, int s, int part) {
    const StagePlan p = stage_plan(h, s);
    if (part >= 0 && (h->limiter || h->sigma > 0.0)) return HYDRO_ESTATE;    // those need the halos before the x sweep
    h->view = part >= 0;
    int rc = eval_stage<R>(h, p.in, p.slot, s, p.c, true, p.w, p.out, p.un, p.a, p.b, part < 0 ? 3 : part == 0 ? 1 : 2);
    h->view = false;
    if (rc != HYDRO_OK) return rc;
    if (s == 2 && part != 0) { h->step += 1; h->prims_valid = false; }   // the next stage 0 refills slot prim_slot
    return HYDRO_OK;
}

template <typename R>
int eval_rhs_impl(hydro* h, double stage_c) {
    int rc;
    if ((rc = ensure_prims<R>(h)) != HYDRO_OK) return rc;
    return eval_stage<R>(h, h->buf[h->cur], h->prim_slot, 0, stage_c, false, 0.0, 0, 0, 0.0, 0.0);
}

template <typename R>
int prims_out_impl(hydro* h, void* out) {
    long long blocks = (h->N + 255) / 256;
    long long cap = (long long)h->num_sms * 8;
    if (blocks > cap) blocks = cap;
    k_prims_out<R><<<(unsigned)blocks, 256, 0, h->stream>>>((const R*)h->buf[h->cur], (R*)out, h->N, h->Np, h->nx, h->nxp, h->nf,
                                                            (R)h->e_floor, (R)(1.0 - h->delta));
    CK(cudaGetLastError());
    return HYDRO_OK;
}

// pitched device buffer (row pitch nxp) -> the caller's dense layout (row length nx), nf*nz*ny rows
int copy_out(hydro* h, const void* dev_src, void* out, int memspace) {
    const cudaMemcpyKind kind = memspace == HYDRO_MEM_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    const size_t row = (size_t)h->nx * h->esz, rows = (size_t)h->nf * h->nz * h->ny;
    if (h->nxp == h->nx) CK(cudaMemcpyAsync(out, dev_src, row * rows, kind, h->stream));
    else CK(cudaMemcpy2DAsync(out, row, dev_src, (size_t)h->nxp * h->esz, row, rows, kind, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return HYDRO_OK;
}

}  // namespace

extern "C" {

int hydro_create(hydro_t** out, int nx, int ny, int nz, double dx, double dt, const hydro_eos_t* eos, void* cuda_stream) {
    if (!out) return HYDRO_EINVAL;
    *out = 0;
    hydro_eos_t o;
    o.eos = HYDRO_EOS_CONFORMAL; o.nfields = 4; o.precision = 64; o.weno_eps = 0; o.v_cap_delta = 0; o.e_floor = 0;
    o.weno_order = 0;
    if (eos) o = *eos;
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dt > 0) || !std::isfinite(dx) || !std::isfinite(dt)) return HYDRO_EINVAL;
    if (o.eos != HYDRO_EOS_CONFORMAL || (o.nfields != 4 && o.nfields != 5) || (o.precision != 64 && o.precision != 32))
        return HYDRO_EINVAL;
    if (o.weno_eps < 0 || o.v_cap_delta < 0 || o.v_cap_delta >= 1 || o.e_floor < 0) return HYDRO_EINVAL;
    if (o.weno_order != 0 && o.weno_order != 5 && o.weno_order != 7) return HYDRO_EINVAL;
    if ((long long)nx * ny * nz > (1LL << 40)) return HYDRO_EINVAL;
    hydro* h = new (std::nothrow) hydro();
    if (!h) return HYDRO_ENOMEM;
    h->nx = nx; h->ny = ny; h->nz = nz; h->nf = o.nfields; h->prec = o.precision;
    h->N = (long long)nx * ny * nz;
    h->order = o.weno_order == 5 ? 5 : 7;
    h->sigma = 0.0;
    h->limiter = 0;
    { const char* ts = getenv("HYDRO_NO_TAIL_SPLIT"); h->tail_split = !(ts && ts[0] == '1'); }
    { const char* ts = getenv("HYDRO_NO_SPLIT5"); h->split5 = !(ts && ts[0] == '1'); }
    h->nz_global = nz; h->k_offset = 0; h->own_lo = 0; h->own_hi = nz;
    h->dx = dx; h->dt = dt;
    h->weno_eps = o.weno_eps > 0 ? o.weno_eps : 1e-6;
    h->delta = o.v_cap_delta > 0 ? o.v_cap_delta : (o.precision == 64 ? 1e-10 : 1e-5);
    h->e_floor = o.e_floor > 0 ? o.e_floor : 1e-12;
    h->esz = o.precision == 64 ? 8 : 4;
    {
        const int per16 = 16 / (int)h->esz;                             // reals per 16 bytes
        h->nxp = (nx + per16 - 1) / per16 * per16;
        h->Np = (long long)h->nxp * ny * nz;
    }
    h->stream = (cudaStream_t)cuda_stream; h->own_stream = false;
    for (int b = 0; b < 3; ++b) h->buf[b] = 0;
    h->cur = 0; h->L = h->P = h->W = 0; h->diag = 0; h->jets_dev = 0;
    h->jets_dirty = false; h->step = 0; h->prim_slot = 0; h->prims_valid = false; h->launches = 0;
    h->profiling = false;
    h->view = false;
    h->graph = 0; h->graph_slot = -1; h->graph_njets = -1; h->graph_launches = 0;
    { const char* ng = getenv("HYDRO_NO_GRAPH"); h->use_graph = !(ng && ng[0] == '1'); }
    h->chain_prev = 0;
    for (int k = 0; k < HYDRO_K_COUNT; ++k) { h->k_ms[k] = 0; h->k_n[k] = 0; }
    int rc = HYDRO_OK;
    do {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) { rc = cuda_fail(h, e, "cudaGetDevice"); break; }
        e = cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) { rc = cuda_fail(h, e, "cudaDeviceGetAttribute"); break; }
        if (!cuda_stream) {
            e = cudaStreamCreateWithFlags(&h->stream, cudaStreamNonBlocking);
            if (e != cudaSuccess) { rc = cuda_fail(h, e, "cudaStreamCreate"); break; }
            h->own_stream = true;
        }
        const size_t fb = (size_t)h->Np * h->nf * h->esz;
        void** ptrs[] = {&h->buf[0], &h->buf[1], &h->buf[2], &h->L};
        for (int b = 0; b < 4 && rc == HYDRO_OK; ++b) {
            e = cudaMalloc(ptrs[b], fb);
            if (e != cudaSuccess) rc = cuda_fail(h, e, "cudaMalloc(state)");
            else if (h->nxp != h->nx && (e = cudaMemsetAsync(*ptrs[b], 0, fb, h->stream)) != cudaSuccess)
                rc = cuda_fail(h, e, "cudaMemset(state)");           // pad columns: finite, never cells
        }
        if (rc != HYDRO_OK) break;
        if ((e = cudaMalloc(&h->P, (size_t)h->Np * h->esz)) != cudaSuccess) { rc = cuda_fail(h, e, "cudaMalloc(P)"); break; }
        if ((e = cudaMalloc(&h->W, (size_t)h->Np * h->esz)) != cudaSuccess) { rc = cuda_fail(h, e, "cudaMalloc(W)"); break; }
        if ((e = cudaMalloc((void**)&h->diag, sizeof(Diag))) != cudaSuccess) { rc = cuda_fail(h, e, "cudaMalloc(diag)"); break; }
        if ((e = cudaMalloc((void**)&h->jets_dev, sizeof(JetDev) * MAX_JETS)) != cudaSuccess) { rc = cuda_fail(h, e, "cudaMalloc(jets)"); break; }
        if ((e = cudaMemsetAsync(h->diag, 0, sizeof(Diag), h->stream)) != cudaSuccess) { rc = cuda_fail(h, e, "cudaMemset(diag)"); break; }
        h->prim_blocks_per_sm = 0;
        if (h->prec == 64) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->prim_blocks_per_sm, k_prim<double>, PRIM_THREADS, 0);
        else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->prim_blocks_per_sm, k_prim<float>, PRIM_THREADS, 0);
        if (e != cudaSuccess || h->prim_blocks_per_sm < 1) h->prim_blocks_per_sm = 2;
        rc = setup_tma(h);
    } while (0);
    if (rc != HYDRO_OK) {
        // keep the error text out of reach of the caller: handle is destroyed
        hydro_destroy(h);
        return rc;
    }
    *out = h;
    return HYDRO_OK;
}

void hydro_destroy(hydro_t* h) {
    if (!h) return;
    if (h->stream || !h->own_stream) cudaStreamSynchronize(h->stream);
    drain_events(h);
    drop_graph(h);
    for (size_t n = 0; n < h->ev_pool.size(); ++n) cudaEventDestroy(h->ev_pool[n]);
    for (int b = 0; b < 3; ++b) cudaFree(h->buf[b]);
    cudaFree(h->L); cudaFree(h->P); cudaFree(h->W); cudaFree(h->diag); cudaFree(h->jets_dev);
    if (h->own_stream && h->stream) cudaStreamDestroy(h->stream);
    delete h;
}

int hydro_set_state(hydro_t* h, const void* U, int memspace) {
    if (!h || !U || (memspace != HYDRO_MEM_HOST && memspace != HYDRO_MEM_DEVICE)) return HYDRO_EINVAL;
    const cudaMemcpyKind kind = memspace == HYDRO_MEM_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    const size_t row = (size_t)h->nx * h->esz, rows = (size_t)h->nf * h->nz * h->ny;
    if (h->nxp == h->nx) CK(cudaMemcpyAsync(h->buf[h->cur], U, row * rows, kind, h->stream));
    else CK(cudaMemcpy2DAsync(h->buf[h->cur], (size_t)h->nxp * h->esz, U, row, row, rows, kind, h->stream));
    CK(cudaMemsetAsync(h->diag, 0, sizeof(Diag), h->stream));
    if (memspace == HYDRO_MEM_HOST) CK(cudaStreamSynchronize(h->stream));
    h->step = 0;
    h->prims_valid = false;
    h->prim_slot = 0;
    for (size_t j = 0; j < h->jets.size(); ++j) h->jets[j].step_added = 0;
    h->jets_dirty = true;
    return HYDRO_OK;
}

int hydro_add_jet(hydro_t* h, double x0, double y0, double z0, double dirx, double diry, double dirz, double kappa_rad,
                  double kappa_coll, double cr_over_cf, int* id) {
    if (!h) return HYDRO_EINVAL;
    const double nrm = std::sqrt(dirx * dirx + diry * diry + dirz * dirz);
    if (!(nrm > 0) || !std::isfinite(nrm) || !std::isfinite(x0 + y0 + z0 + kappa_rad + kappa_coll + cr_over_cf)) return HYDRO_EINVAL;
    if ((int)h->jets.size() >= MAX_JETS) return HYDRO_ESTATE;
    JetDev j;
    j.x0 = x0; j.y0 = y0; j.z0 = z0; j.nx = dirx / nrm; j.ny = diry / nrm; j.nz = dirz / nrm;
    j.k_rad = kappa_rad; j.k_coll = kappa_coll; j.crcf = cr_over_cf; j.step_added = h->step;
    h->jets.push_back(j);
    h->jets_dirty = true;
    if (id) *id = (int)h->jets.size() - 1;
    return HYDRO_OK;
}

// cells of half-width of the Gaussian deposit cube (R15): ceil(3 sigma/dx - 2^-20) clamped to [1, 8]; 0 for the point deposit
static int deposit_radius(const hydro* h, double sigma) {
    if (!(sigma > 0.0)) return 0;
    int r = (int)std::ceil(3.0 * sigma / h->dx - 1.0 / 1048576.0);
    return r < 1 ? 1 : (r > 8 ? 8 : r);
}
static bool is_slab(const hydro* h) { return h->own_lo > 0 || h->own_hi < h->nz; }

int hydro_set_slab(hydro_t* h, int nz_global, int k_offset, int own_lo, int own_hi) {
    if (!h || nz_global < h->nz || k_offset < 0 || k_offset + h->nz > nz_global || own_lo < 0 || own_hi > h->nz || own_lo >= own_hi)
        return HYDRO_EINVAL;
    // an interior slab end must carry the 4 halo planes the stencil needs
    if ((k_offset > 0 && own_lo < 4) || (k_offset + h->nz < nz_global && h->nz - own_hi < 4)) return HYDRO_EINVAL;
    // a Gaussian deposit wider than the halo would lose the part of its cube that a rank cannot see
    if ((own_lo > 0 || own_hi < h->nz) && deposit_radius(h, h->sigma) > 4) return HYDRO_EINVAL;
    h->nz_global = nz_global; h->k_offset = k_offset; h->own_lo = own_lo; h->own_hi = own_hi;
    h->prims_valid = false;
    drop_graph(h);
    return build_map_sets(h, true, own_lo, own_hi);
}

int hydro_stage_prims(hydro_t* h, int s) {
    if (!h || s < 0 || s > 2) return HYDRO_EINVAL;
    return h->prec == 64 ? stage_prims_impl<double>(h, s, -1) : stage_prims_impl<float>(h, s, -1);
}

int hydro_stage_sweeps(hydro_t* h, int s) {
    if (!h || s < 0 || s > 2) return HYDRO_EINVAL;
    return h->prec == 64 ? stage_sweeps_impl<double>(h, s, -1) : stage_sweeps_impl<float>(h, s, -1);
}

int hydro_stage_prims_part(hydro_t* h, int s, int part) {
    if (!h || s < 0 || s > 2 || (part != 0 && part != 1)) return HYDRO_EINVAL;
    return h->prec == 64 ? stage_prims_impl<double>(h, s, part) : stage_prims_impl<float>(h, s, part);
}

int hydro_stage_sweeps_part(hydro_t* h, int s, int part) {
    if (!h || s < 0 || s > 2 || (part != 0 && part != 1)) return HYDRO_EINVAL;
    return h->prec == 64 ? stage_sweeps_impl<double>(h, s, part) : stage_sweeps_impl<float>(h, s, part);
}

int hydro_stage_alpha_dev(hydro_t* h, int s, int set, void* dev_bits) {
    if (!h || s < 0 || s > 2 || !dev_bits) return HYDRO_EINVAL;
    const StagePlan p = stage_plan(h, s);
    unsigned long long* slot_bits = h->diag->slot[p.slot].alpha_bits;
    if (set) CK(cudaMemcpyAsync(slot_bits, dev_bits, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToDevice, h->stream));
    else CK(cudaMemcpyAsync(dev_bits, slot_bits, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToDevice, h->stream));
    return HYDRO_OK;
}

int hydro_stage_alpha(hydro_t* h, int s, int set, double alpha[3]) {
    if (!h || s < 0 || s > 2 || !alpha) return HYDRO_EINVAL;
    const StagePlan p = stage_plan(h, s);
    unsigned long long bits[3];
    if (set) {
        for (int d = 0; d < 3; ++d) {
            if (!(alpha[d] >= 0.0)) return HYDRO_EINVAL;
            if (h->prec == 64) { double x = alpha[d]; memcpy(&bits[d], &x, 8); }
            else { float x = (float)alpha[d]; unsigned int u; memcpy(&u, &x, 4); bits[d] = u; }
        }
        CK(cudaMemcpyAsync(h->diag->slot[p.slot].alpha_bits, bits, sizeof bits, cudaMemcpyHostToDevice, h->stream));
        CK(cudaStreamSynchronize(h->stream));
        return HYDRO_OK;
    }
    CK(cudaMemcpyAsync(bits, h->diag->slot[p.slot].alpha_bits, sizeof bits, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    for (int d = 0; d < 3; ++d) {
        if (h->prec == 64) { double x; memcpy(&x, &bits[d], 8); alpha[d] = x; }
        else { unsigned int u = (unsigned int)bits[d]; float x; memcpy(&x, &u, 4); alpha[d] = x; }
    }
    return HYDRO_OK;
}

int hydro_halo(hydro_t* h, int s, int side, int unpack, void* dev_buf) {
    if (!h || s < 0 || s > 2 || (side != 0 && side != 1) || !dev_buf) return HYDRO_EINVAL;
    // stage s's OUTPUT state (buffer roles are fixed within a handle: buf[cur] = U^n and, after stage 2, U^{n+1})
    char* base = (char*)(s == 0 ? h->buf[(h->cur + 1) % 3] : s == 1 ? h->buf[(h->cur + 2) % 3] : h->buf[h->cur]);
    const size_t plane = (size_t)h->nxp * h->ny * h->esz, width = 4 * plane, fpitch = (size_t)h->Np * h->esz;
    int k0;                                   // first of the 4 planes
    if (!unpack) k0 = side == 0 ? h->own_lo : h->own_hi - 4;            // owned boundary planes -> buffer
    else k0 = side == 0 ? h->own_lo - 4 : h->own_hi;                    // buffer -> halo planes
    if (k0 < 0 || k0 + 4 > h->nz || h->own_hi - h->own_lo < 4) return HYDRO_EINVAL;
    char* planes = base + (size_t)k0 * plane;
    if (!unpack) CK(cudaMemcpy2DAsync(dev_buf, width, planes, fpitch, width, (size_t)h->nf, cudaMemcpyDeviceToDevice, h->stream));
    else CK(cudaMemcpy2DAsync(planes, fpitch, dev_buf, width, width, (size_t)h->nf, cudaMemcpyDeviceToDevice, h->stream));
    return HYDRO_OK;
}

long long hydro_halo_reals(const hydro_t* h) { return h ? (long long)h->nf * 4 * h->ny * h->nxp : -1; }

int hydro_set_limiter(hydro_t* h, int enable) {
    if (!h) return HYDRO_EINVAL;
    if (enable && h->prec != 64) return HYDRO_EINVAL;                  // delta = 1e-8 E is below fp32 resolution
    h->limiter = enable ? 1 : 0;
    drop_graph(h);
    return HYDRO_OK;
}

int hydro_get_limited_faces(hydro_t* h, long long* n) {
    if (!h || !n) return HYDRO_EINVAL;
    Diag d;
    CK(cudaMemcpyAsync(&d, h->diag, sizeof(Diag), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    *n = (long long)d.nlim_total;
    return HYDRO_OK;
}

int hydro_set_deposit_width(hydro_t* h, double sigma) {
    if (!h || !(sigma >= 0.0) || !std::isfinite(sigma)) return HYDRO_EINVAL;
    if (is_slab(h) && deposit_radius(h, sigma) > 4) return HYDRO_EINVAL;          // see hydro_set_slab
    h->sigma = sigma;
    drop_graph(h);
    return HYDRO_OK;
}

int hydro_set_step(hydro_t* h, long long step) {
    if (!h || step < 0) return HYDRO_EINVAL;
    h->step = step;
    CK(cudaMemcpyAsync(&h->diag->step, &h->step, sizeof(long long), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return HYDRO_OK;
}

int hydro_clear_jets(hydro_t* h) {
    if (!h) return HYDRO_EINVAL;
    h->jets.clear();
    h->jets_dirty = true;
    return HYDRO_OK;
}

int hydro_step(hydro_t* h, int nsteps) {
    if (!h || nsteps < 0) return HYDRO_EINVAL;
    h->chain_prev = 0;                                              // other work may sit on the stream since the last launch
    return h->prec == 64 ? step_impl<double>(h, nsteps) : step_impl<float>(h, nsteps);
}

int hydro_synchronize(hydro_t* h) {
    if (!h) return HYDRO_EINVAL;
    CK(cudaStreamSynchronize(h->stream));
    return HYDRO_OK;
}

int hydro_get_fields(hydro_t* h, void* out, int which, int memspace) {
    if (!h || !out || (memspace != HYDRO_MEM_HOST && memspace != HYDRO_MEM_DEVICE)) return HYDRO_EINVAL;
    if (which == HYDRO_FIELDS_CONSERVED) return copy_out(h, h->buf[h->cur], out, memspace);
    if (which != HYDRO_FIELDS_PRIMITIVE) return HYDRO_EINVAL;
    if (memspace == HYDRO_MEM_DEVICE && h->nxp == h->nx) {
        int rc = h->prec == 64 ? prims_out_impl<double>(h, out) : prims_out_impl<float>(h, out);
        if (rc != HYDRO_OK) return rc;
        CK(cudaStreamSynchronize(h->stream));
        return HYDRO_OK;
    }
    // host destination or pitched rows: stage through the RHS buffer (free between steps)
    int rc = h->prec == 64 ? prims_out_impl<double>(h, h->L) : prims_out_impl<float>(h, h->L);
    if (rc != HYDRO_OK) return rc;
    return copy_out(h, h->L, out, memspace);
}

int hydro_eval_rhs(hydro_t* h, double stage_c, void* out, int memspace) {
    if (!h || !out || (memspace != HYDRO_MEM_HOST && memspace != HYDRO_MEM_DEVICE)) return HYDRO_EINVAL;
    int rc = h->prec == 64 ? eval_rhs_impl<double>(h, stage_c) : eval_rhs_impl<float>(h, stage_c);
    if (rc != HYDRO_OK) return rc;
    return copy_out(h, h->limiter ? h->buf[(h->cur + 2) % 3] : h->L, out, memspace);
}

int hydro_get_diag(hydro_t* h, double alpha[3], double* cfl, long long* ncap, int* has_nan, double deposited[4],
                   long long* step) {
    if (!h) return HYDRO_EINVAL;
    Diag d;
    CK(cudaMemcpyAsync(&d, h->diag, sizeof(Diag), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    double am = 0;
    for (int k = 0; k < 3; ++k) {
        if (alpha) alpha[k] = d.alpha_last[k];
        am = d.alpha_last[k] > am ? d.alpha_last[k] : am;
    }
    if (cfl) *cfl = am * h->dt / h->dx;
    if (ncap) *ncap = (long long)d.ncap_total;
    if (has_nan) *has_nan = d.nan_total ? 1 : 0;
    if (deposited) for (int k = 0; k < 4; ++k) deposited[k] = d.deposited[k];
    if (step) *step = h->step;
    return HYDRO_OK;
}

int hydro_get_last_stage_q(hydro_t* h, int jet, double out[3]) {
    if (!h || !out || jet < 0 || jet >= (int)h->jets.size()) return HYDRO_EINVAL;
    Diag d;
    CK(cudaMemcpyAsync(&d, h->diag, sizeof(Diag), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    for (int s = 0; s < 3; ++s) out[s] = d.last_q[s][jet];
    return HYDRO_OK;
}

int hydro_set_profiling(hydro_t* h, int enable) {
    if (!h) return HYDRO_EINVAL;
    CK(cudaStreamSynchronize(h->stream));
    drain_events(h);
    h->profiling = enable != 0;
    if (enable) for (int k = 0; k < HYDRO_K_COUNT; ++k) { h->k_ms[k] = 0; h->k_n[k] = 0; }
    return HYDRO_OK;
}

int hydro_get_kernel_times(hydro_t* h, double ms[HYDRO_K_COUNT], long long launches[HYDRO_K_COUNT]) {
    if (!h) return HYDRO_EINVAL;
    CK(cudaStreamSynchronize(h->stream));
    drain_events(h);
    for (int k = 0; k < HYDRO_K_COUNT; ++k) {
        if (ms) ms[k] = h->k_ms[k];
        if (launches) launches[k] = h->k_n[k];
    }
    return HYDRO_OK;
}

long long hydro_launch_count(const hydro_t* h) { return h ? h->launches : -1; }

int hydro_sweep_path(const hydro_t* h) { return h ? 1 : 0; }

int hydro_measure_alu_peak(int precision, double millis, void* cuda_stream, double* tflops) {
    if (!tflops || (precision != 64 && precision != 32) || !(millis > 0)) return HYDRO_EINVAL;
    hydro* h = 0;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    void* out = 0;
    CK(cudaMalloc(&out, 64));
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    const int blocks = sms * 8, threads = 256;
    int iters = 2000;
    double best = 0, spent = 0;
    for (int rep = 0; rep < 64 && spent < millis; ++rep) {
        cudaEventRecord(a, st);
        if (precision == 64) k_alu_peak<double><<<blocks, threads, 0, st>>>((double*)out, iters, 0.999999, 1e-7);
        else k_alu_peak<float><<<blocks, threads, 0, st>>>((float*)out, iters, 0.9999f, 1e-4f);
        cudaEventRecord(b, st);
        cudaError_t e = cudaEventSynchronize(b);
        if (e != cudaSuccess) { cudaFree(out); return HYDRO_ECUDA; }
        float ms = 0;
        cudaEventElapsedTime(&ms, a, b);
        const double fl = 2.0 * 64.0 * (double)iters * (double)blocks * threads;
        if (rep > 0) { const double tf = fl / (ms * 1e-3) * 1e-12; best = tf > best ? tf : best; spent += ms; }
        if (ms < 2.0f && iters < 400000) iters *= 4;
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    cudaFree(out);
    *tflops = best;
    return HYDRO_OK;
}

const char* hydro_strerror(int code) {
    switch (code) {
        case HYDRO_OK: return "ok";
        case HYDRO_EINVAL: return "invalid argument";
        case HYDRO_ENOMEM: return "out of device memory";
        case HYDRO_ECUDA: return "CUDA error (see hydro_last_cuda_error)";
        case HYDRO_ESTATE: return "invalid state for this call (jet table full, buffer not owned by the handle, or option not available in this precision)";
        default: return "unknown error";
    }
}

const char* hydro_last_cuda_error(const hydro_t* h) { return h ? h->cuda_err.c_str() : ""; }

}  // extern "C"
