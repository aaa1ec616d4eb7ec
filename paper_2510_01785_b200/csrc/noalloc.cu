// cuhpx_ring_weights_noalloc: the ring-weight solver (cuhpx_ring_weights, ring_weights.cu) for callers that cannot
// allocate device memory (code under CUDA graph capture set-up, tight serving loops, harnesses that forbid cudaMalloc).
// Its device scratch -- the tables and ring spectra of the (nside, lmax_w, mmax = 0, fp64) transform plus the
// conjugate-gradient vectors -- lives in the file-scope array below instead of a caller-owned buffer.
//   * CUHPX_NOALLOC_SCRATCH_BYTES (8 MiB, include/cuhpx.h) is the limit: nside <= 512 at the default lmax_w = 3 nside
//     (5.7 MiB); a larger request is refused with CUHPX_EWORKSPACE before anything is launched.
//   * Every GPU that loads libcuhpx.so holds the array until the process exits.
//   * Every call on a device shares it: a call overwrites what the previous one left (everything is cleared first), and
//     two calls whose GPU work overlaps in time (different streams, or different host threads) RACE.  Serialise them.
//   * No cudaMalloc / cudaFree / allocating library call is made here or below; the first call on a device does that
//     device's one-time set-up (the array's address; in the existing path the FFT stage's kernel attributes and its side
//     stream, ring_fft.cu dev_res).
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/cuhpx.h"

// In host code this name is a host-side stand-in for the symbol, NOT a device address: only cudaGetSymbolAddress yields
// the pointer a kernel may use (looked up once per device in scratch_address below).
static __device__ __align__(256) unsigned char cuhpx_noalloc_scratch[CUHPX_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
void* g_addr[MAX_DEVICES];   // device address of cuhpx_noalloc_scratch on device i (null: not looked up yet)

// the array's address on the CURRENT device (each device that loads the module has its own copy)
cudaError_t scratch_address(void** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, cuhpx_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!p || ((uintptr_t)p & 255)) return cudaErrorInvalidSymbol;
        g_addr[dev] = p;
    }
    *out = g_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int cuhpx_ring_weights_noalloc(int nside, int lmax_w, double* d_weights, cuhpx_stream_t stream) {
    const size_t need = cuhpx_ring_weights_workspace_bytes(nside, lmax_w);  // 0: arguments no transform accepts
    if (need == 0 || !d_weights) return CUHPX_EINVAL;
    if (need > (size_t)CUHPX_NOALLOC_SCRATCH_BYTES) return CUHPX_EWORKSPACE;  // beyond the built-in scratch: use cuhpx_ring_weights
    void* scratch = nullptr;
    if (scratch_address(&scratch) != cudaSuccess) return CUHPX_ECUDA;
    // the array keeps the last call's contents: start from zeros (header, tables, spectra, solver vectors and scalars)
    if (cudaMemsetAsync(scratch, 0, need, (cudaStream_t)stream) != cudaSuccess) return CUHPX_ECUDA;
    return cuhpx_ring_weights(nside, lmax_w, d_weights, scratch, (size_t)CUHPX_NOALLOC_SCRATCH_BYTES, stream);
}
