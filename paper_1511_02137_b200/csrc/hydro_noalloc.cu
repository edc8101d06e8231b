// hydro_noalloc.cu -- hydro_wavespeeds_noalloc (include/hydro.h): steps a-1 + a-2 of the path (con2prim for p = e/3, eq. 1
// PAPER.md:17-19, and the exact maxima of the Lax-Friedrichs wavespeeds) of a caller's device state WITHOUT any allocation.
// PRODUCT (sm_100a).  For callers that cannot call cudaMalloc: stream capture, tight serving loops, harnesses that forbid it.
//
// The kernel is the path's own k_prim<double> (hydro_kernels.cuh), unchanged; what differs from hydro_create's handles is
// where its scratch lives: the pressure / inverse-enthalpy arrays it writes (P, W: one real per cell each -- nobody reads
// them here) and the reduction block (Diag) sit in ONE file-scope __device__ array of fixed size instead of cudaMalloc'ed
// buffers.  Every GPU that loads the library holds that array until exit (HYDRO_NOALLOC_MAX_CELLS x 16 bytes + 4 KiB).
// All calls share it and it keeps the last call's contents: the reduction block is cleared at the start of every call (on
// the caller's stream), P and W are overwritten before anything could read them.  Calls that overlap on the GPU (different
// streams, or host threads) RACE on it: serialise them.
#include "../../include/hydro.h"
#include "hydro_kernels.cuh"

#include <cstdio>
#include <mutex>

using namespace hydro_dev;

namespace {

constexpr long long MAX_CELLS = HYDRO_NOALLOC_MAX_CELLS;
constexpr size_t DIAG_BYTES = 4096;                                   // the reduction block, padded
static_assert(sizeof(Diag) <= DIAG_BYTES, "Diag outgrew its slot in the scratch array");
constexpr size_t SCRATCH_BYTES = DIAG_BYTES + 2 * (size_t)MAX_CELLS * sizeof(double);

// In HOST code this name is a host-side stand-in for the symbol, not a device address: never pass it to a kernel.  The
// device address comes from cudaGetSymbolAddress (resolve_device below), once per device, with that device current.
static __device__ __align__(256) unsigned char g_scratch[SCRATCH_BYTES];

struct PerDevice { void* scratch; int num_sms, blocks_per_sm; bool ok; };
PerDevice g_dev[64];
std::mutex g_mu;

void set_err(char* buf, int len, const char* fmt, const char* a = "", long long x = 0, long long y = 0) {
    if (buf && len > 0) snprintf(buf, (size_t)len, fmt, a, x, y);
}

// results out of the reduction block: the bit patterns become doubles, the counters 64-bit integers
__global__ void k_noalloc_finish(const Diag* __restrict__ dg, double* __restrict__ alpha, long long* __restrict__ counts) {
    if (threadIdx.x < 3) alpha[threadIdx.x] = Real<double>::from_bits(dg->slot[0].alpha_bits[threadIdx.x]);
    if (threadIdx.x == 0 && counts) {
        counts[0] = (long long)dg->slot[0].ncap;
        counts[1] = dg->slot[0].nan_flag ? 1 : 0;
    }
}

int resolve_device(int dev, PerDevice** out, char* err, int errlen) {
    if (dev < 0 || dev >= 64) { set_err(err, errlen, "device ordinal out of range%s", ""); return HYDRO_EINVAL; }
    std::lock_guard<std::mutex> lk(g_mu);
    PerDevice& d = g_dev[dev];
    if (!d.ok) {
        void* p = 0;
        cudaError_t e = cudaGetSymbolAddress(&p, g_scratch);          // the device current is `dev` (the caller just asked)
        if (e != cudaSuccess || !p) { set_err(err, errlen, "cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e)); return HYDRO_ECUDA; }
        int sms = 0, bps = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess ||
            (e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_prim<double>, PRIM_THREADS, 0)) != cudaSuccess || bps < 1) {
            set_err(err, errlen, "device query: %s", cudaGetErrorString(e));
            return HYDRO_ECUDA;
        }
        d.scratch = p; d.num_sms = sms; d.blocks_per_sm = bps; d.ok = true;
    }
    *out = &d;
    return HYDRO_OK;
}

}  // namespace

extern "C" int hydro_wavespeeds_noalloc(const void* U_dev, int nx, int ny, int nz, int nfields, double v_cap_delta,
                                        double e_floor, double* alpha_dev, long long* counts_dev, void* cuda_stream,
                                        char* err, int errlen) {
    if (err && errlen > 0) err[0] = 0;
    if (!U_dev || !alpha_dev || nx < 1 || ny < 1 || nz < 1 || (nfields != 4 && nfields != 5)) {
        set_err(err, errlen, "bad argument%s (null pointer, size < 1, or nfields not 4 / 5)", "");
        return HYDRO_EINVAL;
    }
    const long long N = (long long)nx * ny * nz;
    if (N > MAX_CELLS) {
        set_err(err, errlen, "%s%lld cells exceed the fixed scratch of hydro_wavespeeds_noalloc (HYDRO_NOALLOC_MAX_CELLS = %lld)",
                "", N, MAX_CELLS);
        return HYDRO_EINVAL;
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { set_err(err, errlen, "cudaGetDevice: %s", cudaGetErrorString(e)); return HYDRO_ECUDA; }
    PerDevice* pd = 0;
    int rc = resolve_device(dev, &pd, err, errlen);
    if (rc != HYDRO_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned char* base = (unsigned char*)pd->scratch;
    Diag* dg = (Diag*)base;
    double* P = (double*)(base + DIAG_BYTES);
    double* W = P + MAX_CELLS;
    // the array keeps the last call's maxima and counters: they must start at zero
    if ((e = cudaMemsetAsync(dg, 0, sizeof(Diag), st)) != cudaSuccess) {
        set_err(err, errlen, "cudaMemsetAsync: %s", cudaGetErrorString(e));
        return HYDRO_ECUDA;
    }
    PrimArgs<double> a;
    a.U = (const double*)U_dev; a.P = P; a.W = W; a.diag = dg; a.slot = 0;
    a.nx = nx; a.nxp = nx;                                            // the caller's state is dense
    a.c0 = 0; a.N = N; a.Np = N; a.own_lo = 0; a.own_hi = N;
    a.with_alpha = 1; a.seed_slot = 1;                                // a cleared slot: its candidates are cell 0 (valid, clamped)
    a.e_floor = e_floor > 0.0 ? e_floor : 1e-12;                      // hydro_eos_t's defaults (R9)
    a.one_minus_delta = 1.0 - (v_cap_delta > 0.0 ? v_cap_delta : 1e-10);
    long long blocks = (N + PRIM_THREADS - 1) / PRIM_THREADS;
    const long long cap = (long long)pd->num_sms * pd->blocks_per_sm;
    if (blocks > cap) blocks = cap;
    k_prim<double><<<(unsigned)blocks, PRIM_THREADS, 0, st>>>(a);
    k_noalloc_finish<<<1, 32, 0, st>>>(dg, alpha_dev, counts_dev);
    if ((e = cudaGetLastError()) != cudaSuccess) {
        set_err(err, errlen, "kernel launch: %s", cudaGetErrorString(e));
        return HYDRO_ECUDA;
    }
    return HYDRO_OK;
}
