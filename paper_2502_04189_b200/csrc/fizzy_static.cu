// fizzy_static.cu -- fizzy_count_nonfinite_static (include/fizzy.h): the health check of fizzy_check_finite for callers that
// hold nothing but pointers to the fields.  Think of an in-situ monitor or an output plug-in that the solver calls between
// steps: it is handed u, v, w, p, phi, T as device pointers, it owns no fizzy context and no device memory of its own, and
// it may not get any -- the host application has given the whole card to its own pool allocator (a cudaMalloc from a
// plug-in would fail or eat into what the solver was promised), and a cudaMalloc / cudaFree would also stall the solver's
// streams, because both synchronise the device.  So the scratch this reduction needs lives in the library image itself: one
// file-scope __device__ array per GPU that loads libfizzy.so, reserved when the module is loaded and held until the process
// exits.  Nothing in this file calls cudaMalloc, cudaFree or a library routine that allocates device memory.
//
// The kernel is a variant of k_count_nonfinite (fz_diag.cuh).  That one adds per-warp counts into one counter of the
// context's workspace with atomics; this one gives every block a fixed chunk of the index range, lets it write ONE partial
// count into its own slot of the static array, and has the block that finishes last (an atomic ticket) add the slots up in
// slot order.  The number of slots bounds the problem size: see FIZZY_STATIC_MAX_VALUES in fizzy.h.
#include "../../include/fizzy.h"

#include <cstdio>
#include <mutex>

#include <cuda_runtime.h>

namespace {

constexpr int FZS_THREADS = 256;
constexpr int FZS_PER_THREAD = 16;
constexpr int FZS_CHUNK = FZS_THREADS * FZS_PER_THREAD;                        // values of EACH field one block scans
constexpr int FZS_MAX_BLOCKS = (int)(FIZZY_STATIC_MAX_VALUES / FZS_CHUNK);     // 32768 partial-count slots
constexpr int FZS_HEAD = 32;                                                   // words in front of the slots (256 bytes)
static_assert((long long)FZS_MAX_BLOCKS * FZS_CHUNK == FIZZY_STATIC_MAX_VALUES, "the maximum is a whole number of chunks");

// The scratch: word 0 = ticket counter (has to be zero when a launch starts), word 1 = the total the last block leaves
// behind, words FZS_HEAD.. = one partial count per block.  256 KiB + 256 B of device memory on every GPU that loads the
// library.  All calls share it and it keeps whatever the previous call wrote.
static __device__ __align__(256) unsigned long long fzs_scratch[FZS_HEAD + FZS_MAX_BLOCKS];

struct FzsFields {
    const double *f[FIZZY_STATIC_MAX_FIELDS];
    int nf;
};

__device__ __forceinline__ unsigned fzs_block_sum(unsigned v, unsigned *sh)
{
    v = __reduce_add_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    unsigned t = 0;
    if (threadIdx.x < 32) {
        t = threadIdx.x < FZS_THREADS / 32 ? sh[threadIdx.x] : 0u;
        t = __reduce_add_sync(0xffffffffu, t);
    }
    __syncthreads();
    return t;   // valid in warp 0
}

// scr is the DEVICE address of fzs_scratch, looked up by the host with cudaGetSymbolAddress and passed in (device code
// could also name the array directly; the host-side name is only a handle and must never be given to a kernel).
__global__ void __launch_bounds__(FZS_THREADS)
k_count_nonfinite_static(FzsFields F, long long n, unsigned long long *scr)
{
    __shared__ unsigned sh[FZS_THREADS / 32];
    __shared__ bool last;
    const long long base = (long long)blockIdx.x * FZS_CHUNK + threadIdx.x;
    unsigned bad = 0;
    for (int q = 0; q < F.nf; ++q) {
        const double *f = F.f[q];
        unsigned long long bits[FZS_PER_THREAD];
#pragma unroll
        for (int j = 0; j < FZS_PER_THREAD; ++j) {
            const long long i = base + (long long)j * FZS_THREADS;
            bits[j] = i < n ? (unsigned long long)__double_as_longlong(__ldg(f + i)) : 0ull;
        }
#pragma unroll
        for (int j = 0; j < FZS_PER_THREAD; ++j)   // Inf and NaN: all eleven exponent bits set
            bad += (bits[j] & 0x7ff0000000000000ull) == 0x7ff0000000000000ull;
    }
    const unsigned mine = fzs_block_sum(bad, sh);
    if (threadIdx.x == 0) {
        scr[FZS_HEAD + blockIdx.x] = mine;
        __threadfence();                                         // the slot is visible before the ticket is taken
        last = atomicAdd(scr, 1ull) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    // the last block: every slot of this launch is written; slots beyond gridDim.x still hold an older call's counts and
    // are not read
    unsigned long long tot = 0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += FZS_THREADS) tot += __ldcg(scr + FZS_HEAD + b);
    // the total is at most 8 fields x 2^27 values = 2^30: 32-bit partial sums are enough
    const unsigned all = fzs_block_sum((unsigned)tot, sh);
    if (threadIdx.x == 0) {
        scr[1] = all;
        scr[0] = 0ull;                                           // leave the ticket ready for the next launch
    }
}

// Device address of fzs_scratch on each device, looked up once per device (with that device current).
constexpr int FZS_MAX_DEVICES = 64;
std::mutex fzs_mutex;
unsigned long long *fzs_addr[FZS_MAX_DEVICES] = {nullptr};

fizzy_status fzs_fail(fizzy_status s, char *err, size_t err_len, const char *what, const char *detail = nullptr)
{
    if (err && err_len) std::snprintf(err, err_len, "fizzy_count_nonfinite_static: %s%s%s", what, detail ? ": " : "", detail ? detail : "");
    return s;
}

}  // namespace

extern "C" fizzy_status fizzy_count_nonfinite_static(const double *const *dev_fields, int nfields, long long n,
                                                     void *cuda_stream, long long *count, char *err, size_t err_len)
{
    if (err && err_len) err[0] = '\0';
    if (!dev_fields || !count) return fzs_fail(FIZZY_EINVAL, err, err_len, "dev_fields and count must be non-NULL");
    if (nfields < 1 || nfields > FIZZY_STATIC_MAX_FIELDS)
        return fzs_fail(FIZZY_EINVAL, err, err_len, "nfields must be between 1 and FIZZY_STATIC_MAX_FIELDS (8)");
    if (n < 0) return fzs_fail(FIZZY_EINVAL, err, err_len, "n must not be negative");
    if (n > FIZZY_STATIC_MAX_VALUES)
        return fzs_fail(FIZZY_EINVAL, err, err_len,
                        "n exceeds FIZZY_STATIC_MAX_VALUES (2^27 = 134217728 values per field, a 512^3 grid): the built-in "
                        "scratch array has no slot for more; check the fields in pieces or use fizzy_check_finite");
    FzsFields F;
    F.nf = nfields;
    for (int q = 0; q < FIZZY_STATIC_MAX_FIELDS; ++q) F.f[q] = q < nfields ? dev_fields[q] : nullptr;
    for (int q = 0; q < nfields; ++q)
        if (!F.f[q]) return fzs_fail(FIZZY_EINVAL, err, err_len, "a field pointer is NULL");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fzs_fail(FIZZY_ECUDA, err, err_len, "cudaGetDevice", cudaGetErrorString(e));
    if (dev < 0 || dev >= FZS_MAX_DEVICES) return fzs_fail(FIZZY_EINVAL, err, err_len, "device ordinal beyond 63");
    if (n > 0)   // host memory cannot be staged without allocating: the fields must be readable by a kernel on this device
        for (int q = 0; q < nfields; ++q) {
            cudaPointerAttributes pa;
            e = cudaPointerGetAttributes(&pa, F.f[q]);
            if (e != cudaSuccess) { cudaGetLastError(); return fzs_fail(FIZZY_EINVAL, err, err_len, "cudaPointerGetAttributes", cudaGetErrorString(e)); }
            const bool ok = pa.type == cudaMemoryTypeManaged || (pa.type == cudaMemoryTypeDevice && pa.device == dev);
            if (!ok) return fzs_fail(FIZZY_EINVAL, err, err_len, "every field must be device (or managed) memory of the current CUDA device");
        }
    // set-up, once per device: the device address of the scratch array on THIS device
    unsigned long long *scr = nullptr;
    {
        std::lock_guard<std::mutex> lock(fzs_mutex);
        if (!fzs_addr[dev]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, fzs_scratch);
            if (e != cudaSuccess || !p) {
                cudaGetLastError();
                return fzs_fail(FIZZY_ECUDA, err, err_len, "cudaGetSymbolAddress(fzs_scratch)", cudaGetErrorString(e));
            }
            fzs_addr[dev] = static_cast<unsigned long long *>(p);
        }
        scr = fzs_addr[dev];
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (n == 0) { *count = 0; return FIZZY_OK; }
    const unsigned blocks = (unsigned)((n + FZS_CHUNK - 1) / FZS_CHUNK);
    // ticket and total start at zero whatever an earlier (possibly failed) call left there; the slots need no clearing,
    // every slot that is read is written first by this launch
    e = cudaMemsetAsync(scr, 0, 2 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return fzs_fail(FIZZY_ECUDA, err, err_len, "cudaMemsetAsync", cudaGetErrorString(e));
    k_count_nonfinite_static<<<blocks, FZS_THREADS, 0, st>>>(F, n, scr);
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) return fzs_fail(FIZZY_ECUDA, err, err_len, "k_count_nonfinite_static", cudaGetErrorString(e));
    unsigned long long h = 0;
    e = cudaMemcpyAsync(&h, scr + 1, sizeof(h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fzs_fail(FIZZY_ECUDA, err, err_len, "reading the count back", cudaGetErrorString(e));
    *count = (long long)h;
    return FIZZY_OK;
}
