// arc_noalloc.cu -- arc_pix2vec_noalloc: the device HEALPix generator for callers
// that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// The existing entry point arc_pix2vec (arc_run.cu) stages its host arguments in three device buffers that it
// cudaMalloc's and cudaFree's on EVERY call.  This variant stages them in ONE file-scope device array of fixed size
// instead, so the call allocates nothing: no cudaMalloc, no cudaFree, no allocating library routine.
//
//   * The array holds ARC_PIX2VEC_NOALLOC_MAX = 4096 (level, pixel) pairs and their unit vectors:
//     4096 x (4 + 4 + 24) B = 128 KiB.  Every GPU that loads the library holds those 128 KiB until the process exits.
//   * More than 4096 pairs per call is ARC_EINVAL (arc_noalloc_last_error() says so); split the call.
//   * In HOST code the array's name is a host-side stand-in, not a device address: the address is taken once per device,
//     with that device current, by cudaGetSymbolAddress (checked), and that pointer is what the kernel is given.
//   * Every call on a device shares the array, and it keeps the last call's contents.  Nothing in it has to start at
//     zero: a call overwrites the n inputs before the kernel reads them, and the kernel writes the 3 n outputs before
//     they are copied back; entries beyond n are never read.  Calls that overlap on the GPU (two host threads, or a
//     caller that made the copies asynchronous) would race on it: the entry point is synchronous on the legacy default
//     stream and serialised by a mutex, so two calls through it never do.
// Nothing here is shared with oracle/; the arithmetic is arc_pix2vec_dev (arc_healpix.cuh), as in the existing path.
#include <cuda_runtime.h>
#include <stdint.h>
#include <mutex>
#include <string>
#include "../../include/arc.h"
#include "arc_healpix.cuh"

namespace {

constexpr int MAXN = ARC_PIX2VEC_NOALLOC_MAX;
constexpr size_t OFF_LEVEL = 0;                                   // int32_t  [MAXN]
constexpr size_t OFF_PIX = OFF_LEVEL + sizeof(int32_t) * MAXN;    // uint32_t [MAXN]
constexpr size_t OFF_OUT = OFF_PIX + sizeof(uint32_t) * MAXN;     // double   [3 MAXN]  (offset 32 KiB: 256-byte aligned)
constexpr size_t SCRATCH_BYTES = OFF_OUT + sizeof(double) * 3 * MAXN;
static_assert(OFF_OUT % 256 == 0 && SCRATCH_BYTES == 128 * 1024, "scratch layout");

// the scratch memory: file scope, static, in every GPU that loads the library
static __device__ __align__(256) unsigned char arc_noalloc_scratch[SCRATCH_BYTES];

__global__ void __launch_bounds__(128) arc_pix2vec_noalloc_kernel(unsigned char *scratch, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int32_t *level = reinterpret_cast<const int32_t *>(scratch + OFF_LEVEL);
    const uint32_t *pix = reinterpret_cast<const uint32_t *>(scratch + OFF_PIX);
    double *out = reinterpret_cast<double *>(scratch + OFF_OUT);
    double x, y, z;
    arc_pix2vec_dev(level[i], pix[i], x, y, z);
    out[3 * i] = x; out[3 * i + 1] = y; out[3 * i + 2] = z;
}

constexpr int MAX_DEVICES = 64;
std::mutex g_mutex;
unsigned char *g_scratch_ptr[MAX_DEVICES] = {};                   // device address of the array, per device (set-up, once)
thread_local std::string g_err;

int fail(int code, const std::string &msg) { g_err = msg; return code; }

}  // namespace

extern "C" {

int arc_pix2vec_noalloc_max(void) { return MAXN; }

const char *arc_noalloc_last_error(void) { return g_err.c_str(); }

int arc_pix2vec_noalloc(const int32_t *level, const uint32_t *pix, int n, double *out)
{
    if (n < 0 || (n > 0 && (!level || !pix || !out))) return fail(ARC_EINVAL, "arc_pix2vec_noalloc: NULL argument or n < 0");
    if (n > MAXN)
        return fail(ARC_EINVAL, "arc_pix2vec_noalloc: n = " + std::to_string(n) + " exceeds the fixed scratch of " + std::to_string(MAXN) +
                                    " pairs per call (ARC_PIX2VEC_NOALLOC_MAX); split the call or use arc_pix2vec");
    if (n == 0) return ARC_OK;
    for (int i = 0; i < n; ++i)
        if (level[i] < 0 || level[i] > 14 || (unsigned long long)pix[i] >= (12ull << (2 * level[i])))
            return fail(ARC_EINVAL, "arc_pix2vec_noalloc: pair " + std::to_string(i) + " is not a pixel (level in [0, 14], pix < 12 4^level)");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) { cudaGetLastError(); return fail(ARC_ECUDA, "arc_pix2vec_noalloc: no current CUDA device (there is no CPU fallback)"); }
    std::lock_guard<std::mutex> lock(g_mutex);                    // calls share the array: one at a time
    if (!g_scratch_ptr[dev]) {
        // set-up, once per device, with that device current: the array's NAME is a host-side stand-in in host code
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, arc_noalloc_scratch);
        if (e != cudaSuccess || !p) { cudaGetLastError(); return fail(ARC_ECUDA, std::string("arc_pix2vec_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e)); }
        g_scratch_ptr[dev] = static_cast<unsigned char *>(p);
    }
    unsigned char *s = g_scratch_ptr[dev];
    e = cudaMemcpy(s + OFF_LEVEL, level, sizeof(int32_t) * n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(s + OFF_PIX, pix, sizeof(uint32_t) * n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        arc_pix2vec_noalloc_kernel<<<(n + 127) / 128, 128>>>(s, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, s + OFF_OUT, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost);   // (waits for the kernel)
    if (e != cudaSuccess) { cudaGetLastError(); return fail(ARC_ECUDA, std::string("arc_pix2vec_noalloc: ") + cudaGetErrorString(e)); }
    return ARC_OK;
}

}  // extern "C"
